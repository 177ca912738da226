#!/usr/bin/env python
"""Benchmark of the hot path (clip -> dedisperse -> detect) on synthetic BEST-2-shaped filterbanks.

    python bench.py --gpus N --steps K --warmup W [--config 3] [--impl reference]

One "step" = one pass of the whole chain over one buffer of the workload (default: config 3,
8 beams x 1024 channels x 65536 samples fp32, 640 DM trials -- the configuration BASELINE.json's
metric is quoted on).  Prints ONE JSON line (rank 0).  See DESIGN.md section 8 for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

NOMINAL_ADD_PEAK = 148 * 128 * 1.965e9          # SMs x FP32/INT32 lanes x max SM clock (B200_PROFILING.md)
# DRAM bytes of one dedispersion launch from the committed ncu captures (profiles/r1e_*.md); null for other configs
NCU_TRAFFIC_BYTES = {"cfg3-8beam-f32": 17.8e9, "cfg4-8beam-u8": 6.73e9}


def measured_hbm_peak() -> float:
    """HBM bytes/s from the driver-written MEASURED_PEAKS.json, else the profiling guide's fallback figure."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]) * 1e9
    except Exception:
        return 6.65e12          # B200_PROFILING.md fallback


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
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200", "-i", str(self.index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for (ts, line) in self.lines:
            if ts < t0 - 0.1 or ts > t1 + 0.3:
                continue
            f = [s.strip() for s in line.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:   # region shorter than one sample: take the closest sample
            for (ts, line) in self.lines[-3:]:
                f = [s.strip() for s in line.split(",")]
                try:
                    sm.append(float(f[0])); mx.append(float(f[1]))
                except Exception:
                    pass
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(value: float, world: int, device=None) -> float:
    """Max of a per-rank number over the process group (the contract's "max over ranks"); identity at world 1."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank: float, world: int, ms_per_step_rank: float, device=None):
    """Whole-job value: every rank processes its own `units_per_rank` per step (beam sharding, no exchange step),
    the step time is the slowest rank's.  Returns (value, ms_per_step)."""
    ms = max_over_ranks(ms_per_step_rank, world, device)
    return units_per_rank * world / (ms * 1e-3), ms


def oracle_chain_sample(cfg, x_beams):
    """The oracle, as it stands, on a few beams [k][nchans][nsamps] (or one beam [nchans][nsamps]) of the workload:
    clip -> dedisperse (rows) -> detect."""
    import oracle
    t0 = time.perf_counter()
    xb = x_beams.copy()[None] if x_beams.ndim == 2 else x_beams.copy()
    oracle.rfi_clip(xb, cfg.window, cfg.k_chan, cfg.k_spec)
    t1 = time.perf_counter()
    d = oracle.delay_table(cfg.nchans, cfg.f_top, cfg.foff, cfg.tsamp, cfg.dm_low, cfg.dm_step, cfg.ndms)
    out, _ = oracle.dedisperse(xb, d, want_abs=False)
    t2 = time.perf_counter()
    ev, cnt, _ = oracle.detect(out, out.shape[2], cfg.snr_thresh)
    t3 = time.perf_counter()
    units = xb.shape[0] * cfg.ndms * out.shape[2]           # DM-trial samples of the sampled beams
    return units, (t3 - t0), {"clip_s": t1 - t0, "dedisperse_s": t2 - t1, "detect_s": t3 - t2, "events": cnt}


def run_reference(args, cfg):
    """--impl reference: the CPU oracle timed on the host cores, each step one beam of the workload."""
    import oracle
    from workloads import generate_beam
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    x = generate_beam(cfg, 0)
    for _ in range(min(args.warmup, 1)):
        oracle_chain_sample(cfg, x)
    tot_units, tot_t, parts = 0, 0.0, None
    for _ in range(args.steps):
        u, t, parts = oracle_chain_sample(cfg, x)
        tot_units += u
        tot_t += t
    value = tot_units / tot_t
    cores = oracle.num_threads()
    sample = f"1 of {cfg.nbeams} beams of {cfg.name} per step (full clip+dedisperse+detect chain of that beam)"
    line = {
        "impl": "reference", "metric": "DM-trial samples/s", "value": value, "unit": "DM-trial samples/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * tot_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64" if cfg.dtype == "f32" else "u32",
        "data": "synthetic", "config": {"workload": cfg.name, "sample": sample},
        "cpu_baseline": {"value": value, "unit": "DM-trial samples/s", "cores": cores, "kind": "oracle", "sample": sample,
                         "stage_seconds": parts},
        "e2e": {"value": value, "unit": "DM-trial samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", type=int, default=0, help="dedisp_kernel option: 0 auto, 1 direct, 2 tiled")
    ap.add_argument("--geom", type=int, default=-1, help="tiled_geom_<dtype> option (compiled tile geometry); -1 = plan default")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--nstreams", type=int, default=8)
    ap.add_argument("--pairs", type=int, default=-1, help="plan option pair_presum (fp32: exact channel-pair pre-sums); -1 = plan default")
    ap.add_argument("--postprocess", type=int, default=0,
                    help="median window W: also time mdsm_median_filter(W) + mdsm_detrend on the dedispersed series (fp32 "
                         "configs; reported beside the chain, not part of `value`)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    from workloads import CONFIGS, generate
    cfg = CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist

    import paper_1307_5700_b200 as m

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # ---- workload: every rank owns its own buffer of the same shape (beam sharding, no collective) ----
    import dataclasses
    cfg_r = dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank)
    x = generate(cfg_r)
    torch_dt = torch.float32 if cfg.dtype == "f32" else torch.uint8
    h_in = torch.from_numpy(x).pin_memory()
    pristine = h_in.cuda(non_blocking=False)
    work = torch.empty_like(pristine)
    plan = m.mdsm_plan_create(*cfg.plan_args())
    m.mdsm_plan_set_option(plan, "dedisp_kernel", args.kernel)
    if args.pairs >= 0:
        m.mdsm_plan_set_option(plan, "pair_presum_u8" if cfg.dtype == "u8" else "pair_presum", args.pairs)
    if args.geom >= 0:
        m.mdsm_plan_set_option(plan, "tiled_geom_" + cfg.dtype, args.geom)
    nso = m.mdsm_plan_nsamps_out(plan)
    out = torch.empty((cfg.nbeams, cfg.ndms, cfg.nsamps), dtype=torch.float32 if cfg.dtype == "f32" else torch.int32,
                      device="cuda")
    max_events = 1 << 22
    events = torch.empty((max_events, 4), dtype=torch.int32, device="cuda")
    count = torch.zeros(1, dtype=torch.int64, device="cuda")
    out_dtype = m.MDSM_F32 if cfg.dtype == "f32" else m.MDSM_U8
    stream = torch.cuda.current_stream()

    def step(evs=None):
        work.copy_(pristine)                       # restore the un-clipped input (also flushes L2: 2.1 GB > 126 MB)
        count.zero_()
        if evs: evs[0].record(stream)
        m.mdsm_rfi_clip(plan, work, 0, cfg.nbeams, cfg.window, cfg.k_chan, cfg.k_spec, None, None, stream)
        if evs: evs[1].record(stream)
        m.mdsm_dedisperse(plan, work, 0, cfg.nbeams, out, stream)
        if evs: evs[2].record(stream)
        m.mdsm_detect(plan, out, 0, cfg.nbeams, cfg.snr_thresh, events, max_events, count, stream, dtype=out_dtype)
        if evs: evs[3].record(stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    l0 = m.mdsm_plan_launch_count(plan)
    barrier()
    t0 = time.time()
    for i in range(args.steps):
        step(evs[i])
    barrier()
    t1 = time.time()
    launches = m.mdsm_plan_launch_count(plan) - l0
    clocks = sampler.stop(t0, t1)
    n_events = int(count.item())
    clip_ms = [e[0].elapsed_time(e[1]) for e in evs]
    dd_ms = [e[1].elapsed_time(e[2]) for e in evs]
    det_ms = [e[2].elapsed_time(e[3]) for e in evs]
    chain_ms = [e[0].elapsed_time(e[3]) for e in evs]
    value, ms_per_step = job_throughput(cfg.nbeams * cfg.ndms * nso, world, sum(chain_ms) / args.steps, "cuda")
    units_per_step = cfg.nbeams * cfg.ndms * nso * world

    # ---- optional: the paper's post-processing stage, timed on the series of the last step ----
    post = None
    if args.postprocess and cfg.dtype == "f32":
        filt = torch.empty_like(out)
        pe = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        tm, td = [], []
        for _ in range(max(3, min(args.steps, 10))):
            work.copy_(pristine)                                   # L2 flush between repetitions
            pe[0].record(stream)
            m.mdsm_median_filter(plan, out, filt, 0, cfg.nbeams, args.postprocess, stream)
            pe[1].record(stream)
            m.mdsm_detrend(plan, filt, 0, cfg.nbeams, None, stream)
            pe[2].record(stream)
            torch.cuda.synchronize()
            tm.append(pe[0].elapsed_time(pe[1])); td.append(pe[1].elapsed_time(pe[2]))
        sbytes = 4.0 * cfg.nbeams * cfg.ndms * nso
        hp = measured_hbm_peak()
        post = {"median_window": args.postprocess, "median_ms": statistics.mean(tm), "detrend_ms": statistics.mean(td),
                "median_hbm_frac": 2 * sbytes / (statistics.mean(tm) * 1e-3) / hp,
                "detrend_hbm_frac": 2 * sbytes / (statistics.mean(td) * 1e-3) / hp,
                "algorithmic_bytes": "one read + one write of the valid series per kernel"}
        del filt
        # the paper's first GPU stage (power from 16-bit complex voltages, NEXT-4) on a buffer of the input's shape
        nel = cfg.nbeams * cfg.nchans * cfg.nsamps
        volt = torch.randint(-2048, 2048, (nel, 2), dtype=torch.int16, device="cuda")
        tp = []
        for _ in range(5):
            out.zero_()                                            # 1.3 GB write: flushes L2
            pe[0].record(stream)
            m.mdsm_power_i16(volt, work, nel, stream)
            pe[1].record(stream)
            torch.cuda.synchronize()
            tp.append(pe[0].elapsed_time(pe[1]))
        post["power_ms"] = statistics.mean(tp[1:])
        post["power_hbm_frac"] = 8.0 * nel / (post["power_ms"] * 1e-3) / hp
        del volt
        # mu-law quantiser (Eq. 5, NEXT-4) on the fp32 input buffer (power is non-negative: use |x|)
        src = work.abs_()
        codes = torch.empty((nel,), dtype=torch.uint8, device="cuda")
        xmax = torch.zeros(1, dtype=torch.float32, device="cuda")
        tq = []
        for _ in range(5):
            out.zero_()
            pe[0].record(stream)
            m.mdsm_mulaw_u8(src, codes, nel, 255.0, xmax, stream)
            pe[1].record(stream)
            torch.cuda.synchronize()
            tq.append(pe[0].elapsed_time(pe[1]))
        post["mulaw_ms"] = statistics.mean(tq[1:])
        post["mulaw_hbm_frac"] = 9.0 * nel / (post["mulaw_ms"] * 1e-3) / hp
        del codes

    # ---- end to end through the host-buffer C-ABI call (H2D of the input and D2H of the events inside) ----
    e2e = None
    if not args.no_e2e:
        h_events = np.zeros(max_events, dtype=m.EVENT_DTYPE)
        for _ in range(2):
            m.mdsm_pipeline_host(plan, h_in, cfg.window, cfg.k_chan, cfg.k_spec, cfg.snr_thresh, h_events, max_events,
                                 args.nstreams)
        barrier()
        l1 = m.mdsm_plan_launch_count(plan)
        te = time.perf_counter()
        n_e2e = max(3, min(args.steps, 10))
        for _ in range(n_e2e):
            rc, cnt_h = m.mdsm_pipeline_host(plan, h_in, cfg.window, cfg.k_chan, cfg.k_spec, cfg.snr_thresh, h_events,
                                             max_events, args.nstreams)
        barrier()
        te = (time.perf_counter() - te) / n_e2e
        te = max_over_ranks(te, world, "cuda")
        launches_e2e = (m.mdsm_plan_launch_count(plan) - l1) // n_e2e
        e2e = {"value": units_per_step / te, "unit": "DM-trial samples/s", "h2d_bytes_per_step": int(x.nbytes),
               "d2h_bytes_per_step": int(cnt_h * 16 + 8), "ms_per_step": 1e3 * te, "events": cnt_h,
               "nstreams": args.nstreams, "gpu_launches_per_step": int(launches_e2e), "timer": "host perf_counter around the call"}

    # ---- roofline of the dominant kernel (dedispersion): issued-add bound, measured peak in this run ----
    peaks = {"fadd": m.mdsm_measure_add_peak(0), "fadd2": m.mdsm_measure_add_peak(1), "iadd": m.mdsm_measure_add_peak(2)}
    peak = max(peaks["fadd"], peaks["fadd2"]) if cfg.dtype == "f32" else peaks["iadd"]
    dd = statistics.mean(dd_ms) * 1e-3
    adds = float(cfg.nchans) * cfg.nbeams * cfg.ndms * nso          # algorithmic adds per launch
    hbm_bytes = x.nbytes + 4.0 * cfg.nbeams * cfg.ndms * nso
    hbm_peak = measured_hbm_peak()
    roofline = {"bound": "alu", "kernel": "dedisperse (mdsm_dedisperse call: pre-pass or widening kernel + tiled kernel, timed together)", "achieved": adds / dd / 1e9, "peak": peak / 1e9, "unit": "Gadd/s",
                "frac": adds / dd / peak, "peak_source": "measured in this run: mdsm_measure_add_peak (register-only add loop, all SMs)",
                "peak_nominal": NOMINAL_ADD_PEAK / 1e9, "measured_peaks_gadd_s": {k: v / 1e9 for k, v in peaks.items()},
                "ms_per_launch": dd * 1e3, "hbm_floor_ms": 1e3 * hbm_bytes / hbm_peak, "traffic": NCU_TRAFFIC_BYTES.get(cfg.name),
                "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of one launch, ncu --set full capture under profiles/ (r1i fp32: pre-pass 6.7 GB + tiled kernel 11.1 GB; r1k u8: pre-pass 2.77 GB + tiled kernel 3.96 GB)"}

    line = {
        "metric": "DM-trial samples/s", "value": value, "unit": "DM-trial samples/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
        "config": {"workload": cfg.name, "nbeams_per_gpu": cfg.nbeams, "nchans": cfg.nchans, "nsamps": cfg.nsamps,
                   "ndms": cfg.ndms, "chain": "rfi_clip+dedisperse+detect", "snr_thresh": cfg.snr_thresh,
                   "l2": "input restored from a pristine 2.1 GB copy before every step (larger than L2)",
                   "dedisp_kernel": args.kernel, "tiled_geom": args.geom},
        "realtime_beams_640dm": cfg.nbeams * world * nso * cfg.tsamp / (ms_per_step * 1e-3),
        "stage_ms": {"rfi_clip": statistics.mean(clip_ms), "dedisperse": statistics.mean(dd_ms), "detect": statistics.mean(det_ms)},
        "dedisperse_only": {"value": units_per_step / world / dd, "unit": "DM-trial samples/s"},
        "events_per_step": n_events, "gpu_launches": int(launches), "clocks": clocks,
        "e2e": e2e, "roofline": roofline,
    }
    if post:
        line["postprocess"] = post

    if rank == 0 and not args.no_cpu_baseline and world >= 1:
        import oracle
        nsample = min(cfg.nbeams, 4)
        u, t, parts = oracle_chain_sample(cfg, x[:nsample])
        line["cpu_baseline"] = {"value": u / t, "unit": "DM-trial samples/s", "cores": oracle.num_threads(), "kind": "oracle",
                                "sample": f"beams 0..{nsample - 1} of {cfg.nbeams} of {cfg.name}, full chain, {t:.1f} s", "stage_seconds": parts}
    m.mdsm_plan_destroy(plan)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
