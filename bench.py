#!/usr/bin/env python
"""bench.py -- FDAS hot path throughput on B200 (contract: see DESIGN.md "Measurement").

A step = one pass of the whole hot path over one DM trial of the SKA config
(BASELINE.json configs[2]: 2^23 samples, 85 templates, width 256, segment 2048):
fdas_spectrum -> fdas_correlate (full f-fdot plane in HBM) -> fdas_harmsum (1..16 harmonics,
merged candidate list).  `value` = DM trials/s with the series resident in HBM; `e2e` = the
same through fdas_search_host with pinned HOST buffers (H2D of the series and D2H of the
candidate list inside the timed region).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "DM trials/s (2^23 samples, 85 z; spectrum + f-fdot plane + 16-harmonic sum)"
UNIT = "DM trials/s"
FP32_LANES_PER_SM = 128                                 # Blackwell guide: 4 sub-partitions x 32 FP32 lanes


def fp32_peak_tflops(n_sms=148, sm_mhz=1965.0):
    """Plain-ALU FP32 peak: SMs x 128 lanes x 2 flop (FMA) x clock.  Defaults are the B200's
    148 SMs and clocks.max.sm; run_ours() passes the SM count the device reports and, separately, the clock
    sampled under load."""
    return n_sms * FP32_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12


FP32_PEAK_TFLOPS = fp32_peak_tflops()


def committed_traffic(kernel_substr):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the kernel whose name contains
    `kernel_substr`, from the committed ncu summary profiles/ncu_dram_bytes.csv (kernel,read,write); None if no
    capture has been committed (bench.py never runs under a profiler)."""
    path = os.path.join(ROOT, "profiles", "ncu_dram_bytes.csv")
    try:
        for line in open(path):
            f = [c.strip() for c in line.split(",")]
            if len(f) >= 3 and kernel_substr in f[0] and f[1].replace(".", "").isdigit():
                return float(f[1]) + float(f[2])
    except OSError:
        pass
    return None


def workload_flops(info):
    """Algorithmic flops of the fused correlate kernel per DM trial (SURVEY.md §8(d) convention:
    5 L log2 L per complex FFT, 6 per complex multiply, 3 per power)."""
    L, m, n_t, n_bins = info.seg_len, info.width, info.n_templates, info.n_bins
    n_seg = math.ceil(n_bins / (L - m + 1))       # the minimum segmentation at this L, m (the library's step L - m gives one more)
    return n_seg * (5 * L * math.log2(L) * (1 + n_t) + 6 * L * n_t) + 3 * n_t * n_bins


class ClockSampler:
    """Samples nvidia-smi SM clocks / throttle reasons during the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = sorted(int(r[0]) for r in self.rows if len(r) >= 6 and r[0].isdigit())
        mx = [int(r[1]) for r in self.rows if len(r) >= 6 and r[1].isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 6 and r[2 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def host_description():
    """CPU model and the oracle's compiler flags, for the cpu_baseline record."""
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    import oracle
    return {"cpu_model": model, "nproc": os.cpu_count(), "oracle_cflags": " ".join(getattr(oracle, "CFLAGS", []))}


def oracle_sample(cfg, x, frac_log2=4):
    """Time the oracle, as it stands, on a bounded sample of one DM trial: the full O1 spectrum, then
    O7 overlap-save correlation + O6 harmonic sum on the first n_bins/2^frac_log2 bins; extrapolate."""
    import oracle
    T = oracle.templates(cfg.z_max, cfg.dz, cfg.width)           # init stage, untimed (as on the GPU)
    thr = oracle.thresholds(16)
    t0 = time.perf_counter()
    S, _ = oracle.spectrum(x)
    t1 = time.perf_counter()
    nb = cfg.n_bins >> frac_log2
    P = oracle.correlate_fft(S[:nb], T, cfg.seg_len)
    t2 = time.perf_counter()
    oracle.harmsum(P, 16, thr)
    t3 = time.perf_counter()
    mult = 1 << frac_log2
    t_dm = (t1 - t0) + mult * ((t2 - t1) + (t3 - t2))
    return t_dm, {"spectrum_s": t1 - t0, "correlate_fft_s": (t2 - t1) * mult, "harmsum_s": (t3 - t2) * mult,
                  "cores": oracle.n_threads(),
                  "sample": "1 DM trial: full O1 spectrum + O7 FFT correlation and O6 harmonic sum on the first "
                            "1/%d of the bins, scaled x%d" % (mult, mult)}


def run_reference(args):
    """--impl reference: the oracle on the host cores (rank 0 only), each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1511_07343_b200 import synth
    import oracle
    oracle.build()
    cfg = synth.config(2)
    x = cfg.series()
    times, detail = [], None
    for i in range(args.warmup + args.steps):
        t_dm, detail = oracle_sample(cfg, x, frac_log2=4)
        if i >= args.warmup:
            times.append(t_dm)
    t = sum(times) / len(times)
    val = 1.0 / t
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[2] (SKA beam, single DM) + configs[4] harmonic sum",
                   "n_samples": cfg.n_samples, "n_z": cfg.n_z, "width": cfg.width, "segment_len": cfg.seg_len},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": detail["cores"], "kind": "oracle",
                         "sample": detail["sample"], **host_description()},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def run_sweep(args):
    """--sweep-templates: the paper's one experiment (Fig. 2), execution time against the
    number of templates for one 2^23-sample series: spectrum + fused correlate with the plane stored, for
    21 ... 121 templates (z_max = n_t - 1, dz = 2, width 256, segment 2048).  One JSON line."""
    import torch
    from paper_1511_07343_b200 import build as fbuild, fdas, synth
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    fbuild.build()
    cfg = synth.config(2)
    d_x = torch.from_numpy(cfg.series()).cuda().view(1, -1)
    stream = torch.cuda.current_stream()
    rows = []
    for n_t in (21, 41, 61, 85, 101, 121):
        plan = fdas.Plan(cfg.n_samples, float(n_t - 1), 2.0, cfg.width, cfg.seg_len)
        d_spec, d_mu, d_plane = plan.empty_spectrum(1), torch.empty(1, device="cuda"), plan.empty_plane(1)

        def step():
            fdas.fdas_spectrum(plan.handle, d_x, 1, d_spec, d_mu, plan.workspace)
            fdas.fdas_correlate(plan.handle, d_spec, 1, d_plane, 0.0, None, None, 0)
        for _ in range(max(3, args.warmup)):
            step()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(args.steps):
            step()
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        rows.append({"n_templates": n_t, "ms_per_dm": ms, "dm_trials_per_s": 1e3 / ms,
                     "plane_outputs_per_s": n_t * plan.info.n_bins / (ms * 1e-3),
                     "frac_of_fft_roofline": (workload_flops(plan.info) + 2.5 * cfg.n_samples * math.log2(cfg.n_samples))
                     / (FP32_PEAK_TFLOPS * 1e12) / (ms * 1e-3)})
        plan.close()
        del d_plane
    print(json.dumps({"sweep_templates": rows, "n_samples": cfg.n_samples, "width": cfg.width,
                      "segment_len": cfg.seg_len, "steps": args.steps, "data": "synthetic",
                      "note": "the plane (n_t x 2^22 fp32) is written every step: larger than L2 from 8 templates on"}))


def run_ab(args):
    """--ab: time the tuning keys (FDAS_OPT_TUNE_*) in one process: fused correlate scalar / packed and its
    template chunking, harmonic sum for several sector counts and tile shapes.  One JSON line; nothing here
    is a bench value."""
    import torch
    from paper_1511_07343_b200 import build as fbuild, fdas, synth
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    fbuild.build()
    cfg = synth.config(2)
    plan = fdas.Plan(cfg.n_samples, cfg.z_max, cfg.dz, cfg.width, cfg.seg_len)
    d_x = torch.from_numpy(cfg.series()).cuda().view(1, -1)
    d_spec, d_mu = plan.spectrum(d_x)
    d_plane = plan.empty_plane(1)
    cap = 1 << 22
    cands = plan.empty_cands(cap)
    thr = fdas.thresholds(16)
    stream = torch.cuda.current_stream()

    def timed(fn, opts):
        for k, v in opts.items():
            fdas.fdas_plan_set_option(plan.handle, k, v)
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(args.steps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        for k in opts:
            fdas.fdas_plan_set_option(plan.handle, k, 0)
        return e0.elapsed_time(e1) / args.steps

    corr = lambda: fdas.fdas_correlate(plan.handle, d_spec, 1, d_plane, 0.0, None, None, 0)
    spec = lambda: fdas.fdas_spectrum(plan.handle, d_x, 1, d_spec, d_mu, plan.workspace)
    hs = lambda: fdas.fdas_harmsum(plan.handle, d_plane[0], 16, thr, cands[0], cands[1], cap)
    out = {"spectrum_ms": {}, "correlate_ms": {}, "harmsum_ms": {}, "steps": args.steps, "plan_status": plan.status()}
    F = fdas
    for name, opts in (("tma_3pass", {}), ("generic_2pass", {F.FDAS_OPT_TUNE_SPEC_GENERIC: 1})):
        out["spectrum_ms"][name] = timed(spec, opts)
    spec()
    for name, opts in (("packed", {}), ("scalar", {F.FDAS_OPT_TUNE_SCALAR: 1}),
                       ("packed_1chunk", {F.FDAS_OPT_TUNE_T_CHUNKS: 1}), ("packed_2chunks", {F.FDAS_OPT_TUNE_T_CHUNKS: 2}),
                       ("packed_4chunks", {F.FDAS_OPT_TUNE_T_CHUNKS: 4}), ("packed_6chunks", {F.FDAS_OPT_TUNE_T_CHUNKS: 6}),
                       ("staged_4seg", {F.FDAS_OPT_TUNE_STAGE_TEMPLATES: 1}),
                       ("staged_4seg_1chunk", {F.FDAS_OPT_TUNE_STAGE_TEMPLATES: 1, F.FDAS_OPT_TUNE_T_CHUNKS: 1})):
        out["correlate_ms"][name] = timed(corr, opts)
    corr()
    for name, opts in (("S16", {}), ("S1", {F.FDAS_OPT_TUNE_HS_SECTORS: 1}), ("S8", {F.FDAS_OPT_TUNE_HS_SECTORS: 8}),
                       ("S32", {F.FDAS_OPT_TUNE_HS_SECTORS: 32}), ("S64", {F.FDAS_OPT_TUNE_HS_SECTORS: 64}),
                       ("S16_1warp", {F.FDAS_OPT_TUNE_HS_ROWS: 1}),
                       ("S16_8warps", {F.FDAS_OPT_TUNE_HS_ROWS: 8}), ("S16_128col", {F.FDAS_OPT_TUNE_HS_VARIANT: 1}),
                       ("S32_128col", {F.FDAS_OPT_TUNE_HS_VARIANT: 1, F.FDAS_OPT_TUNE_HS_SECTORS: 32})):
        out["harmsum_ms"][name] = timed(hs, opts)
        out.setdefault("harmsum_candidates", {})[name] = int(cands[1][0])
    print(json.dumps(out))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1511_07343_b200 import build as fbuild, fdas, shard, synth

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        fbuild.build()
    if world > 1:
        dist.barrier()
    fdas.lib()
    n_sms = torch.cuda.get_device_properties(local).multi_processor_count
    global FP32_PEAK_TFLOPS
    FP32_PEAK_TFLOPS = fp32_peak_tflops(n_sms)

    cfg = synth.config(2)
    n_rot = 4                                   # distinct resident series rotated per step: 134 MB > 126 MB L2
    cap = 1 << 22
    plan = fdas.Plan(cfg.n_samples, cfg.z_max, cfg.dz, cfg.width, cfg.seg_len)
    info = plan.info
    base = cfg.series()                         # seeded series with the 8 injected signals
    host = torch.empty((n_rot, cfg.n_samples), dtype=torch.float32).pin_memory()
    my_dms = shard.dm_shard(n_rot * world, rank, world)     # global DM-trial indices of this rank (dm mod world)
    for r, dm in enumerate(my_dms):             # independent noise per DM trial (seed per DM), same 8 signals
        host[r] = torch.from_numpy(base if dm == 0 else
                                   synth.make_series(cfg.n_samples, cfg.series_seed(dm), cfg.signals[0]))
    d_series = host.cuda()
    d_spec = plan.empty_spectrum(1)
    d_mu = torch.empty(1, dtype=torch.float32, device="cuda")
    d_plane = plan.empty_plane(1)
    cands = plan.empty_cands(cap)
    thr = fdas.thresholds(16)
    stream = torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step(i, marks=None):
        x = d_series[i % n_rot].view(1, -1)
        if marks is not None: marks[0].record(stream)
        fdas.fdas_spectrum(plan.handle, x, 1, d_spec, d_mu, plan.workspace)
        if marks is not None: marks[1].record(stream)
        fdas.fdas_correlate(plan.handle, d_spec, 1, d_plane, 0.0, None, None, 0)
        if marks is not None: marks[2].record(stream)
        fdas.fdas_harmsum(plan.handle, d_plane[0], 16, thr, cands[0], cands[1], cap)
        if marks is not None: marks[3].record(stream)

    for i in range(args.warmup):
        step(i)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    marks = [[ev() for _ in range(4)] for _ in range(args.steps)]
    torch.cuda.synchronize()
    e0, e1 = ev(), ev()
    e0.record(stream)
    for i in range(args.steps):
        step(args.warmup + i, marks[i])
    e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = e0.elapsed_time(e1)
    stage_all = np.array([[m[j].elapsed_time(m[j + 1]) for j in range(3)] for m in marks])
    stage = stage_all.mean(axis=0)
    fp32_measured, _ = fdas.fdas_measure_fp32_tflops()       # FFMA-chain microbenchmark (untimed region)
    fp32_packed, _ = fdas.fdas_measure_fp32_tflops(packed=True)
    l2_gbs = fdas.fdas_measure_l2_gbs()                      # L2 -> SM read bandwidth (untimed region)
    n_found = int(cands[1][0])
    assert plan.status() & fdas.FDAS_STATUS_COPY_TIMEOUT == 0, "an asynchronous copy timed out in the timed region (fdas_plan_status)"

    # BASELINE.json configs[3] (streaming batch, plane not stored, threshold fused into the segment kernel):
    # a batch of 8 resident DM trials per call, spectrum + fused correlate, reported beside the headline
    nb3 = 8
    plan3 = fdas.Plan(cfg.n_samples, cfg.z_max, cfg.dz, cfg.width, cfg.seg_len, max_batch=nb3)
    d_series3 = d_series.repeat(nb3 // n_rot, 1).contiguous()
    d_spec3 = plan3.empty_spectrum(nb3)
    d_mu3 = torch.empty(nb3, dtype=torch.float32, device="cuda")
    cands3 = plan3.empty_cands(1 << 16, n_batch=nb3)

    def step3():
        fdas.fdas_spectrum(plan3.handle, d_series3, nb3, d_spec3, d_mu3, plan3.workspace)
        fdas.fdas_correlate(plan3.handle, d_spec3, nb3, None, 20.0, cands3[0], cands3[1], 1 << 16)
    for _ in range(2):
        step3()
    k3 = max(2, args.steps // 4)
    f0, f1 = ev(), ev()
    torch.cuda.synchronize()
    f0.record(stream)
    for _ in range(k3):
        step3()
    f1.record(stream)
    torch.cuda.synchronize()
    fused_ms = f0.elapsed_time(f1) / (k3 * nb3)
    fused_found = int(cands3[1].sum())
    plan3.close()
    del d_series3, d_spec3, cands3

    # end to end through the host-buffer entry point: pinned host series in, candidate lists out.  One call
    # searches a batch of n_e2e DM trials (the n_rot series, repeated) and overlaps the copy of series i+1
    # with the kernels of series i inside the library (PAPER.md:49 step 1); every series is copied
    # host->device and every candidate list device->host inside the timed region.
    n_e2e = max(4, min(args.steps, 16))
    host_e2e = torch.empty((n_e2e, cfg.n_samples), dtype=torch.float32).pin_memory()
    for i in range(n_e2e):
        host_e2e[i] = host[i % n_rot]
    e2e_cap = 1 << 20
    h_c = torch.zeros((n_e2e, e2e_cap, 3), dtype=torch.int32).pin_memory()
    h_n = torch.zeros(n_e2e, dtype=torch.int32).pin_memory()
    plan.search_host(host_e2e, 16, thr, e2e_cap, h_c, h_n)          # warm-up: allocates the arena, streams, events
    torch.cuda.synchronize()
    e2e_rep = 2
    t0 = time.perf_counter()
    for _ in range(e2e_rep):
        plan.search_host(host_e2e, 16, thr, e2e_cap, h_c, h_n)
    e2e_ms = (time.perf_counter() - t0) * 1e3 / (e2e_rep * n_e2e)
    counts = h_n.numpy().astype(np.int64)
    assert (counts <= e2e_cap).all() and counts.min() > 0, "e2e candidate lists overflowed or empty"
    d2h = int(counts.mean()) * 12 + 4
    clocks = sampler.stop() if rank == 0 else None

    t = torch.tensor([ms, e2e_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms, e2e_ms = float(t[0]), float(t[1])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    ms_step = ms / args.steps
    value = world * 1e3 / ms_step
    flops = workload_flops(info)
    spec_ms, corr_ms, hs_ms = (float(v) for v in stage)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    hbm_src = "MEASURED_PEAKS.json hbm_gbs (of measured)" if "hbm_gbs" in peaks else "6650 GB/s (of fallback, B200_PROFILING.md)"
    plane_bytes = 4 * info.n_templates * info.n_bins
    corr_tf = flops / (corr_ms * 1e-3) / 1e12
    kernels = {
        "spectrum": {"kernels": "k_spec_cols (pass A, pass B) + k_spec_scale + k_spec_rows (pass C): TMA-staged", "bound": "hbm", "ms": spec_ms,
                     "algorithmic_bytes": 4 * cfg.n_samples + 8 * info.n_bins,
                     "achieved": (4 * cfg.n_samples + 8 * info.n_bins) / (spec_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s"},
        "correlate": {"kernels": "k_correlate_2048", "bound": "alu", "ms": corr_ms, "algorithmic_flops": flops,
                      "achieved": corr_tf, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                      "peak_measured_ffma": fp32_measured, "frac_of_measured_ffma": corr_tf / fp32_measured,
                      "hbm_side": {"bytes": plane_bytes + 8 * info.n_bins,
                                   "achieved_gbs": (plane_bytes + 8 * info.n_bins) / (corr_ms * 1e-3) / 1e9, "peak_gbs": hbm_peak}},
        "harmsum": {"kernels": "k_harmsum<5,4,3>", "bound": "hbm", "ms": hs_ms, "algorithmic_bytes": plane_bytes,
                    "l2_to_sm_bytes_inherent": 5.84 * plane_bytes,    # sum over the 16 streams of (h/16)^2
                    "l2_measured_gbs": l2_gbs, "frac_of_l2_stream_bound": 5.84 * plane_bytes / (hs_ms * 1e-3) / 1e9 / l2_gbs,
                    "achieved": plane_bytes / (hs_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s"},
    }
    for k in kernels.values():
        k["frac"] = k["achieved"] / k["peak"]
    dom = max(kernels, key=lambda n: kernels[n]["ms"])          # the kernel with the largest share of the step
    kd = kernels[dom]
    roofline = {"kernel": dom + " (" + kd["kernels"] + ")", "bound": kd["bound"], "achieved": kd["achieved"],
                "peak": kd["peak"], "unit": kd["unit"], "frac": kd["frac"],
                "traffic": committed_traffic({"spectrum": "k_spec", "correlate": "k_correlate", "harmsum": "k_harmsum"}[dom]),
                "ms_per_launch": kd["ms"], "share_of_step": kd["ms"] / (spec_ms + corr_ms + hs_ms),
                "peak_source": hbm_src if kd["bound"] == "hbm" else
                "derived: %d SMs (queried) x 128 FP32 lanes x 2 x 1.965 GHz clocks.max.sm (DESIGN.md section 6)" % n_sms,
                "per_unit": "bytes: the plane read once (4 n_t n_bins)" if dom == "harmsum" else
                "flops: SURVEY 8(d) convention, bench.py::workload_flops" if dom == "correlate" else "bytes: series + spectrum"}
    # north_star's FFT-correlation roofline for spectrum + correlate: the slower of flops at FP32 peak and bytes at HBM peak
    fft_flops = flops + 2.5 * cfg.n_samples * math.log2(cfg.n_samples)
    fft_bytes = 4 * cfg.n_samples + plane_bytes
    t_roof_ms = max(fft_flops / (FP32_PEAK_TFLOPS * 1e12), fft_bytes / (hbm_peak * 1e9)) * 1e3
    t_roof3_ms = max(fft_flops / (FP32_PEAK_TFLOPS * 1e12), 4 * cfg.n_samples / (hbm_peak * 1e9)) * 1e3   # no plane bytes
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[2] (SKA beam, single DM: 2^23 samples, 85 templates, width 256, "
                               "segment 2048, full plane stored) + configs[4] harmonic sum (1..16) on that plane",
                   "n_samples": cfg.n_samples, "n_z": info.n_z, "width": info.width, "segment_len": info.seg_len,
                   "dm_trials_per_step": 1, "l2": "4 resident series rotated (134 MB) and a 1.43 GB plane written "
                                                  "per step: inputs exceed the 126 MB L2",
                   "parallelism": "DM trials sharded across ranks, no collective"},
        "plane_outputs_per_s": world * info.n_templates * info.n_bins / (corr_ms * 1e-3),
        "stage_ms": {"spectrum": spec_ms, "correlate": corr_ms, "harmsum": hs_ms},
        "stage_ms_median": dict(zip(("spectrum", "correlate", "harmsum"), (float(v) for v in np.median(stage_all, axis=0)))),
        "stage_ms_min": dict(zip(("spectrum", "correlate", "harmsum"), (float(v) for v in stage_all.min(axis=0)))),
        "fp32_peak": {"nominal_tflops": FP32_PEAK_TFLOPS, "n_sms": n_sms, "measured_ffma_tflops": fp32_measured,
                      "measured_ffma2_tflops": fp32_packed,
                      "at_sampled_clock_tflops": fp32_peak_tflops(n_sms, clocks["sm_mhz"]) if clocks and clocks.get("sm_mhz") else None},
        "fft_correlation_roofline": {"ms_at_roofline": t_roof_ms, "ms_measured": spec_ms + corr_ms,
                                     "frac": t_roof_ms / (spec_ms + corr_ms),
                                     "dm_trials_per_s_without_harmsum": world * 1e3 / (spec_ms + corr_ms)},
        "fused_batch": {"workload": "BASELINE.json configs[3]: %d resident DM trials per call, spectrum + correlate with "
                                    "the threshold (20) fused, plane not stored" % nb3,
                        "ms_per_dm": fused_ms, "dm_trials_per_s": world * 1e3 / fused_ms,
                        "frac_of_fft_roofline": t_roof3_ms / fused_ms, "candidates_found": fused_found},
        "candidates_found": n_found,
        "occupancy": {k: dict(zip(("ctas_per_sm", "registers", "smem_bytes"), fdas.fdas_kernel_occupancy(k))) for k in fdas.OCCUPANCY_KERNELS},
        "gpu_launches": 6 * args.steps,        # 4 spectrum kernels + fused correlate + harmonic sum (+ 1 memset node)
        "plan_status": plan.status(),
        "clocks": clocks,
        "e2e": {"value": world * 1e3 / e2e_ms, "unit": UNIT, "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": cfg.n_samples * 4, "d2h_bytes_per_step": d2h,
                "how": "fdas_search_host on %d pinned series per call, x%d calls" % (n_e2e, e2e_rep)},
        "roofline": roofline,
        "kernels": kernels,
    }
    if world == 1 and not args.no_cpu:
        import oracle
        oracle.build()
        t_dm, d = oracle_sample(cfg, base, frac_log2=4)
        out["cpu_baseline"] = {"value": 1.0 / t_dm, "unit": UNIT, "cores": d["cores"], "kind": "oracle",
                               "sample": d["sample"], "spectrum_s": d["spectrum_s"],
                               "correlate_fft_s": d["correlate_fft_s"], "harmsum_s": d["harmsum_s"], **host_description()}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--ab", action="store_true", help="time the kernel variants kept for tuning instead")
    ap.add_argument("--sweep-templates", action="store_true",
                    help="time spectrum + correlate against the number of templates (PAPER.md Fig. 2) instead")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.gpus > 1 and "RANK" not in os.environ and args.impl == "ours" and not (args.ab or args.sweep_templates):
        # not under torchrun: start one rank per GPU ourselves (the driver's own launch line does the same)
        port = 29500 + os.getpid() % 2000
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if args.ab:
        run_ab(args)
    elif args.sweep_templates:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
