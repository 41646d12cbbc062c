#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path (beamform+de-dispersion -> inverse PPF -> trigger) on
synthetic LOFAR-shaped data, per the driver contract.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config i | --all-configs]
                    [--mode series|trigger_only|causal|lsmr|exact] [--parallel replicas|beams] [--impl reference]

A step is one lofar_run_block over one block of the workload (default: BASELINE.json:configs[2], the
24 stations x 488 sub-bands x 24 beams case the north_star target names).  `value` is reconstructed
5 ns samples/s per beam with the input resident in HBM; `e2e` is the same through lofar_stream_push
with the blocks in pinned HOST memory (H2D inside the timed region, candidates/sigma copied back); for
configs[4] the e2e leg is the configuration BASELINE.json states: 10 consecutive blocks of 195312 slices.
`--mode` selects the rows "next" of SURVEY.md 8(f): trigger_only (series == NULL), causal (sigma of the
previous block, series-free), lsmr (LSMR inversion, 25 iterations), exact (paper-order de-dispersion).
N > 1: `--parallel replicas` (default; north_star: no sharding or collectives -> N independent replicas, weak
scaling) or `--parallel beams` (f4: the beams are split over the ranks and every step starts with an NCCL
broadcast of the input block from rank 0; strong scaling).  `--gpus N` without a torchrun environment
re-launches itself under torch.distributed.run.
`--impl reference` times the CPU oracle on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import platform
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1612_06592_b200 import shard, synth  # noqa: E402

METRIC = "reconstructed 5 ns samples/s per beam"
UNIT = "samples/s/beam"
MODES = ("series", "trigger_only", "causal", "lsmr", "exact")


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_summary():
    """dram traffic / limiter per kernel from the committed ncu post-processing (profile_summary.py)."""
    path = os.path.join(ROOT, "profiles", "ncu_summary.json")
    if os.path.exists(path):
        return json.load(open(path))
    return {}


def workload(idx: int, slices: int | None):
    w = synth.config(idx)
    if slices:
        from dataclasses import replace
        w = replace(w, T=slices)
    return w


def describe(w, extra=None):
    d = {"workload": f"configs[{w.index}] {w.name}: S={w.S} pols=2 B={w.B} D={w.D} K={w.K} (k0={w.k0}) "
                     f"T={w.T} slices/block {w.dtype}",
         "stations": w.S, "beams": w.B, "trials": w.D, "subbands": w.K, "slices_per_block": w.T,
         "input_dtype": w.dtype, "block_seconds_of_data": w.T * w.slice_seconds,
         "l2": "inputs larger than L2 (no flush needed)" if w.input_bytes > 256e6 else "L2 flushed between steps"}
    if extra:
        d.update(extra)
    return d


# ------------------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[2:6]):
                if v.strip().lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_model() -> str:
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return platform.processor() or "unknown"


# ------------------------------------------------------------------------------------- oracle legs
def oracle_pipe(oracle, w, tau, mode):
    kw = {}
    if mode == "lsmr":
        kw = dict(inversion="lsmr", lsmr_iters=25)
    elif mode == "exact":
        kw = dict(dedisp="exact")
    elif mode == "causal":
        kw = dict(sigma_mode="causal")
    return oracle.OraclePipeline(tau=tau, stec=np.asarray(w.stec), K=w.K, k0=w.k0, kappa=w.kappa, **kw)


def oracle_sample(w, X_sample, tau, budget_s=15.0, mode="series", threads=None):
    """Times the oracle as it stands on a bounded sample (the first `nq` slices of the block, all
    stations/sub-bands/beams/trials); returns (samples/s/beam, cores, description, seconds)."""
    from oracle import lofar_oracle as oracle
    if threads:
        oracle.set_threads(threads)
    pipe = oracle_pipe(oracle, w, tau, mode)
    nq = 8
    t0 = time.perf_counter()
    pipe.run_block(np.ascontiguousarray(X_sample[:, :, :, :nq]))
    probe = time.perf_counter() - t0
    per_slice = max(probe / nq, 1e-6)
    nq = int(min(X_sample.shape[3], max(8, budget_s / per_slice))) // 8 * 8
    pipe.reset()
    xs = np.ascontiguousarray(X_sample[:, :, :, :nq])
    t0 = time.perf_counter()
    pipe.run_block(xs)
    dt = time.perf_counter() - t0
    return nq * w.M / dt, oracle.threads(), f"first {nq} slices of one block, all {w.nseries} series", dt


def cpu_baseline(w, X, tau, mode, budget_s=10.0):
    from oracle import lofar_oracle as oracle
    ncores = os.cpu_count() or 1
    v, cores, sample, dt = oracle_sample(w, X, tau, budget_s, mode, threads=ncores)
    v1, _, sample1, dt1 = oracle_sample(w, X, tau, budget_s / 2, mode, threads=1)
    oracle.set_threads(ncores)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "seconds": dt,
            "single_thread": {"value": v1, "cores": 1, "sample": sample1, "seconds": dt1},
            "cpu_model": cpu_model(), "build": oracle.BUILD_FLAGS,
            "note": "oracle/ as it stands (fp64, naive O(M*K) inverse DFT, direct convolution); a reported baseline, "
                    "not the target"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workload(args.config, args.slices)
    _, _, tau = synth.geometry(w)
    from dataclasses import replace
    ws = replace(w, T=min(w.T, 2048))
    X = synth.generate_block(ws, 0, tau=tau)
    vals, cores, sample = [], 1, ""
    budget = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for i in range(args.warmup + args.steps):
        v, cores, sample, dt = oracle_sample(w, X, tau, budget, args.mode)
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([dt for _, dt in vals]) * 1e3)
    from oracle import lofar_oracle as oracle
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded, paper_1612_06592_b200.synth)",
        "config": describe(w, {"mode": args.mode, "note": "each step is a bounded sample of the block"}),
        "real_time_factor": value / 200e6,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "cpu_model": cpu_model(), "build": oracle.BUILD_FLAGS},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ------------------------------------------------------------------------------------- replicas
def max_over_ranks(value: float, dist, device="cpu") -> float:
    """MAX over ranks of a per-rank duration (the contract's multi-GPU timing rule)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(samples_per_block: int, world: int, ms_step_max: float) -> float:
    """Whole-job samples/s per beam with replicas: every replica reconstructs its own block per step."""
    return world * samples_per_block / (ms_step_max * 1e-3)


def configure_mode(binding, plan, mode):
    if mode == "lsmr":
        plan.set_inversion(binding.LOFAR_INV_LSMR, 25)
    elif mode == "exact":
        plan.set_dedispersion(binding.LOFAR_DEDISP_EXACT)
    elif mode == "causal":
        plan.set_sigma_mode(binding.LOFAR_SIGMA_CAUSAL)


# ------------------------------------------------------------------------------------- GPU arm
def run_gpu(args, idx=None):
    import torch
    from paper_1612_06592_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            dist.init_process_group("nccl")
    binding.load()
    mode = args.mode
    beams_sharded = world > 1 and args.parallel == "beams"

    w = workload(args.config if idx is None else idx, args.slices)
    _, _, tau = synth.geometry(w)
    b0, b1 = shard.beam_slice(w.B, world, rank) if beams_sharded else (0, w.B)
    from dataclasses import replace
    wl = replace(w, B=b1 - b0)                               # what this rank computes
    X = synth.generate_block(w, 0, tau=tau) if (not beams_sharded or rank == 0) else None
    plan = binding.plan_for(wl, tau[b0:b1])
    cap = 4096
    plan.set_trigger(w.kappa, 1, cap)
    configure_mode(binding, plan, mode)
    if args.overlap:
        plan.set_overlap(1, args.overlap_chunk)              # two-lane pipeline (measured slower; off by default)
    if args.scratch_mb:
        plan.set_scratch_limit(args.scratch_mb << 20)        # e.g. an L2-sized beam-sum chunk
    want_series = mode in ("series", "lsmr", "exact")
    Xd = torch.from_numpy(X).cuda() if X is not None else torch.empty((w.S, 2, w.K, w.T, 2),
                                                                       dtype=torch.int8 if w.dtype == "ci8" else torch.int16,
                                                                       device="cuda")
    if want_series:
        series, cand, count, sigma = binding.new_outputs(plan, w.T)
    else:
        series, (cand, count, sigma) = None, binding.new_outputs(plan, 0)[1:]
    stream = torch.cuda.current_stream()
    flush = None
    if w.input_bytes <= 256e6:                               # small inputs: evict them from L2 between steps
        flush = torch.empty(192 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    fl = []

    def step(timed=False):
        if flush is not None:                                # timed separately and subtracted from the step time
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); flush.fill_(1); b.record(stream)
            if timed:
                fl.append((a, b))
        if beams_sharded:
            shard.broadcast_input(Xd, dist, 0)               # the one collective of the sharded path
        plan.run_block(Xd, w.T, series, cand, count, sigma, stream)

    for _ in range(args.warmup):
        step()
    barrier()
    plan.profile(True)
    plan.profile_read()
    l0 = plan.launch_count()
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step(timed=True)
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1) - sum(a.elapsed_time(b) for a, b in fl)
    clocks = sampler.stop() if sampler else None
    launches = plan.launch_count() - l0
    kms, kn = plan.profile_read()
    plan.profile(False)
    ms_total = max_over_ranks(ms_total, dist, "cuda")
    ms_step = ms_total / args.steps
    n_cand = int(count.item())

    # ---- e2e: the same through lofar_stream_push from pinned host memory
    stream_cfg4 = w.index == 4 and args.slices is None
    nbuf = 2 if stream_cfg4 else 1
    Xh = [torch.from_numpy(X if X is not None else np.zeros((w.S, 2, w.K, w.T, 2), dtype=w.np_dtype)).pin_memory()]
    if nbuf == 2:
        Xh.append(torch.from_numpy(synth.generate_block(w, 1, tau=tau)).pin_memory())
    cand_h = torch.zeros((cap, 24), dtype=torch.uint8).pin_memory()
    count_h = torch.zeros(1, dtype=torch.int32).pin_memory()
    sigma_h = torch.zeros(wl.nseries, dtype=torch.float32).pin_memory()
    e2e_steps = w.blocks if stream_cfg4 else max(3, min(args.steps, 5))
    e2e = None
    if not beams_sharded:
        plan.stream_reset()
        for i in range(2):
            plan.stream_push(Xh[i % nbuf], w.T, series, cand_h, count_h, sigma_h)
        plan.stream_sync(allow=(binding.LOFAR_E_OVERFLOW,))
        if stream_cfg4:
            plan.stream_reset()
        barrier()
        t0 = time.perf_counter()
        for i in range(e2e_steps):
            plan.stream_push(Xh[i % nbuf], w.T, series, cand_h, count_h, sigma_h)
        plan.stream_sync(allow=(binding.LOFAR_E_OVERFLOW,))
        torch.cuda.synchronize()
        e2e_s = max_over_ranks(time.perf_counter() - t0, dist, "cuda")
        e2e_ms = e2e_s / e2e_steps * 1e3
        e2e_value = aggregate_value(w.T * w.M, world, e2e_ms)
        e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(w.input_bytes),
               "d2h_bytes_per_step": int(4 + 4 * wl.nseries + cap * 24), "ms_per_step": e2e_ms,
               "real_time_factor": e2e_value / world / 200e6, "steps": e2e_steps,
               "h2d_GBps": w.input_bytes / 1e9 / (e2e_ms * 1e-3),
               "api": "lofar_stream_push + lofar_stream_sync (pinned host input, double-buffered)",
               "note": ("configs[4] as stated: 10 consecutive blocks of 195312 slices, sustained; the blocks alternate "
                        "between two pinned staging buffers generated before the timed region (91.5 GB of distinct "
                        "blocks are not pinned; SURVEY 8(d) allows it)") if stream_cfg4 else
                       "the same block pushed repeatedly"}

    if rank != 0:
        if dist is not None and idx is None:
            dist.destroy_process_group()
        return

    samples_per_block = w.T * w.M
    if beams_sharded:
        value = samples_per_block / (ms_step * 1e-3)          # all B beams of one block per step, over N GPUs
    else:
        value = aggregate_value(samples_per_block, world, ms_step)
    peak, peak_src = peaks()

    # algorithmic bytes per launch group
    esz = 4 if w.dtype == "ci16" else 2
    B, ns = wl.B, wl.nseries
    ninv = B if mode == "exact" else ns
    out_series = want_series and mode not in ("lsmr", "exact")
    by_kernel = [
        ("beamform", w.S * 2 * w.K * w.T * esz + B * w.K * w.T * 8),
        ("ippf_kernel", B * w.K * w.T * 8 + (ninv * w.T * w.M * 4 if (out_series or mode in ("lsmr", "exact")) else 0)),
        ("trigger", ns * (w.T // 16) * 12 + (2 * ns * w.T * w.M * 4 if mode in ("lsmr", "exact") else 0)),
        ("lsmr (25 iterations)", ninv * w.T * w.M * 4 * (8 + 11 * 25)),      # per iteration: v pass 3, u pass 3 + h/hbar/x 4 or 6
        ("dedisp_kernel", (B * 16 / 14 + ns) * w.T * w.M * 4),
    ]
    tc = w.dtype == "ci8" and B >= 4 and w.S <= 32
    shown = {"beamform": "beamform_tc_kernel" if tc else "beamform_kernel"}
    kernels = []
    for i, (nme, nbytes) in enumerate(by_kernel):
        if kn[i] == 0:
            continue
        ms_all = kms[i] / args.steps                          # all launches of this group in one step
        per_step = max(1, int(kn[i]) // args.steps)
        kernels.append({"kernel": shown.get(nme, nme), "launches_per_step": per_step,
                        "ms_per_step": ms_all, "ms_per_launch": ms_all / per_step,
                        "share_of_step": ms_all / ms_step,
                        "algorithmic_GB_per_launch": nbytes / 1e9 / per_step,
                        "achieved_GBps": nbytes / 1e9 / (ms_all * 1e-3)})
    dom = max(kernels, key=lambda k: k["ms_per_step"])
    chain_bytes = w.input_bytes + (ns * w.T * w.M * 4 if want_series else 0)
    prof = ncu_summary().get(f"configs[{w.index}]", {}).get(dom["kernel"], {})
    traffic = None
    if prof.get("dram_GB_per_launch") and prof.get("algorithmic_GB_per_launch") and mode == "series" and args.slices is None:
        traffic = dom["algorithmic_GB_per_launch"] * prof["dram_GB_per_launch"] / prof["algorithmic_GB_per_launch"]
    roofline = {"kernel": dom["kernel"], "bound": "hbm", "achieved": dom["achieved_GBps"], "peak": peak,
                "unit": "GB/s", "frac": dom["achieved_GBps"] / peak, "traffic": traffic,
                "traffic_unit": "GB per launch: ncu dram__bytes_read.sum + dram__bytes_write.sum scaled to this launch "
                                "(profiles/ncu_summary.json)" if traffic else None,
                "limiter": prof.get("limiter"), "fp32_pipe_frac": prof.get("fma_pipe_frac"),
                "issue_frac": prof.get("issue_frac"),
                "algorithmic_GB_per_launch": dom["algorithmic_GB_per_launch"],
                "ms_per_launch": dom["ms_per_launch"], "peak_source": peak_src,
                "note": "achieved = algorithmic bytes per launch / mean launch duration, CUDA events on the "
                        "launching stream inside the timed region (K*8 B read + 4096 B written per series-slice "
                        "for ippf_kernel; 2*S*2*esize B read + B*8 B written per (sub-band, slice) for beamform). "
                        "`bound` names the roofline the kernel is designed against; `limiter` is what ncu shows."}
    # The same kernel against the fp32 pipe (configs 2-4 are predicted ALU-bound): flop per (series, slice)
    # of the inverse PPF = 512-point complex FFT, 5 N log2 N = 23040 (the usual count, twiddles included) + pair pre-pass
    # 8 flop x 256 pairs = 2048 + FIR 2 x 16 taps x 1024 = 32768 -> 57856; peak = SMs x 128 FMA lanes x 2 flop x the SM
    # clock sampled during the timed region.
    if dom["kernel"] == "ippf_kernel":
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        mhz = (clocks or {}).get("sm_mhz") or 1965.0
        flop = 57856.0 * ninv * w.T / dom["launches_per_step"]
        if mode in ("lsmr",):
            flop -= 32768.0 * ninv * w.T / dom["launches_per_step"]          # no FIR in the kernel: LSMR solves instead
        peak_tf = sms * 128 * 2 * mhz * 1e6 / 1e12
        ach_tf = flop / (dom["ms_per_launch"] * 1e-3) / 1e12
        roofline["alu"] = {"bound": "alu", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach_tf / peak_tf,
                           "flop_per_series_slice": 57856,
                           "note": "fp32 pipe: SMs x 128 lanes x 2 flop x sampled SM clock; what ncu names as the busiest "
                                   "units is in `limiter`"}
    chain = {"algorithmic_GB_per_step": chain_bytes / 1e9,
             "achieved_GBps": chain_bytes / 1e9 / (ms_step * 1e-3),
             "frac_of_peak": chain_bytes / 1e9 / (ms_step * 1e-3) / peak,
             "note": "whole chain: input read once + series written once (SURVEY 8(d) fused count); "
                     "series-free modes: input only"}

    # cuFFT (through torch.fft.irfft), timed ONLY as a comparison for step a3 (north_star); never on the product path.
    cufft = None
    if args.compare_cufft and world == 1:
        nb = min(w.nseries * w.T, 1 << 19)                       # slices per batch (4 GB of spectra + 2 GB out)
        spec = torch.zeros((nb, 513), dtype=torch.complex64, device="cuda")
        spec[:, w.k0:w.k0 + w.K] = torch.randn((nb, w.K), dtype=torch.complex64, device="cuda")
        for _ in range(2):
            y = torch.fft.irfft(spec, n=1024, dim=1, norm="forward")
        torch.cuda.synchronize()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        for _ in range(5):
            y = torch.fft.irfft(spec, n=1024, dim=1, norm="forward")
        c1.record()
        torch.cuda.synchronize()
        ms = c0.elapsed_time(c1) / 5
        cufft = {"what": "torch.fft.irfft (cuFFT C2R, 1024 points) on dense 513-bin spectra already transposed to "
                         "slice-major; no beam-sum transpose, no FIR, no trigger sums", "slices": nb,
                 "ns_per_slice": ms * 1e6 / nb, "ms_scaled_to_block": ms * (w.nseries * w.T) / nb,
                 "ippf_kernel_ns_per_slice": next(k["ms_per_step"] for k in kernels if k["kernel"] == "ippf_kernel")
                 * 1e6 / (w.nseries * w.T)}
        del spec, y

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(w, X[:, :, :, :2048], tau, mode)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "strong" if beams_sharded else "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic (seeded, paper_1612_06592_b200.synth)",
        "config": describe(w, {"mode": mode, "pipeline": ("two-lane (lofar_plan_set_overlap 1)" if args.overlap else "serial"),
                               "chunks": [list(c) for c in plan.chunks(w.T)][:3] + ["..."] if len(plan.chunks(w.T)) > 3
                               else [list(c) for c in plan.chunks(w.T)],
                               "parallelism": ("beams sharded over ranks, input broadcast (NCCL)"
                                                             if beams_sharded else "replicas only") if world > 1
                               else "single GPU"}),
        "real_time_factor": (value if beams_sharded else value / world) / 200e6,
        "aggregate_samples_per_s_all_series": value * w.nseries,
        "candidates_last_step": n_cand,
        "e2e": e2e if e2e is not None else {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                                           "note": "beam-sharded run: no streaming leg"},
        "gpu_launches": int(launches),
        "roofline": roofline, "kernels": kernels, "chain": chain,
        "cpu_baseline": cpu, "clocks": clocks, "cufft_comparison": cufft,
    }
    print(json.dumps(line), flush=True)
    plan.destroy()
    if dist is not None and idx is None:
        dist.destroy_process_group()


def relaunch_under_torchrun(args):
    """`--gpus N` by itself: become N ranks (one per GPU) under torch.distributed.run."""
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json:configs (default 2)")
    ap.add_argument("--all-configs", action="store_true", help="one JSON line per config 0..4 (same schema)")
    ap.add_argument("--mode", default="series", choices=MODES)
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "beams"])
    ap.add_argument("--slices", type=int, default=None, help="override slices per block (debugging)")
    ap.add_argument("--impl", default="gpu", choices=["gpu", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--overlap", action="store_true",
                    help="lofar_plan_set_overlap(1): beamformer of chunk c+1 beside the inverse PPF of chunk c")
    ap.add_argument("--overlap-chunk", type=int, default=0, help="slices per pipeline chunk (0 = library default)")
    ap.add_argument("--scratch-mb", type=int, default=0, help="lofar_plan_set_scratch_limit in MiB (0 = default 16 GiB)")
    ap.add_argument("--compare-cufft", action="store_true", help="also time cuFFT C2R (via torch) as a comparison for a3")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "gpu":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_under_torchrun(args)
    if args.all_configs:
        for i in range(len(synth.CONFIGS)):
            run_gpu(args, idx=i)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
