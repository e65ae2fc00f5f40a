#!/usr/bin/env python
"""bench.py - throughput of the SFT inner-product hot path on B200 (driver contract in DESIGN.md §8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

One "step" = one pass of the whole hot path (waveform -> bin selection -> kernel coefficients ->
response -> contraction -> reduction over SFTs) over one batch of synthetic
input: ``sft_inner_products`` for the full template bank of the workload.  Default workload:
BASELINE.json configs[1] ("config2-F": ET-like BNS bank, 4096 templates x 10,800 SFT slots, 10 %
gaps, K = +-8 bins, Fresnel kernel, 0PN+1PN, complex64 data), the config the metric is quoted on.

metric  = active template-SFT(-channel) pairs per second, whole job (sum over ranks / max time).
value   : inputs resident in HBM, device-side CUDA-event time per step, L2 flushed between steps.
e2e     : same call with HOST buffers (pinned params in, results out) through the C ABI; the
          host<->device copies are inside the timed region.
roofline: the fused main kernel against the ALU bound derived in DESIGN.md §7.
cpu_baseline / --impl reference: the fp64 oracle (oracle/, as it stands) on the host cores, on a
          bounded sample of the same workload.

Under torchrun (N > 1) every rank runs the same data store with its own template shard (weak
scaling, no data-path collective: templates are independent).
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "template-SFT inner products/s (<x,h>,<h,h>)"
UNIT = "template-SFT pairs/s"


# ---------------------------------------------------------------------------------------------
def make_workload(name, rank=0, n_templates=None, n_sft=None, K=None):
    from paper_2502_11823_b200 import workloads as wl
    if name == "config1":
        return wl.config1(n_templates=n_templates or 64)
    if name == "config2":
        kw = dict(n_templates=n_templates or 4096, bank_seed=5 + 1000 * rank)
        if n_sft:
            kw["n_sft"] = n_sft
        if K is not None:
            kw["K"] = K
        return wl.config2(**kw)
    if name == "config3":
        return wl.config3(n_templates=n_templates or 16384, bank_seed=6 + 1000 * rank)
    if name == "config4":
        return wl.config4(n_templates=n_templates or 65536)
    raise SystemExit("unknown workload %r" % name)


def oracle_objects(w):
    from oracle import inner as oin
    plan = oin.Plan(**w.desc)
    store = oin.Store(bins=w.bins.astype(np.complex128), psd_scale=w.psd_scale, psd_shape=w.psd_shape,
                      response=None if w.response is None else w.response.astype(np.complex128))
    return oin, plan, store


def cores_used():
    """--impl reference runs the oracle in this process: single-threaded numpy elementwise code (no BLAS call on its hot
    path), so 1; the number of host cores available is reported beside it."""
    return 1


_ORACLE = {}


def _oracle_init(desc, bins, psd_scale, psd_shape, response):
    from oracle import inner as oin
    _ORACLE["oin"] = oin
    _ORACLE["plan"] = oin.Plan(**desc)
    _ORACLE["store"] = oin.Store(bins=bins.astype(np.complex128), psd_scale=psd_scale, psd_shape=psd_shape,
                                 response=None if response is None else response.astype(np.complex128))


def _oracle_rows(rows):
    r = _ORACLE["oin"].inner_products(_ORACLE["plan"], _ORACLE["store"], rows)
    return int((r["kc"] >= 0).sum())


def time_oracle(w, budget_s=12.0, seed=99):
    """Times oracle.inner.inner_products (as it stands: numpy fp64, one call per block of templates) on a seeded sample of
    the workload's templates, spread over the host cores with one worker process per core (the oracle itself is
    single-threaded elementwise numpy).  The sample is sized from a one-template probe so that the run takes about
    ``budget_s`` seconds.  Returns (pairs/s, templates, seconds, active pairs, worker processes)."""
    import multiprocessing as mp
    oin, plan, store = oracle_objects(w)
    t0 = time.perf_counter()
    oin.inner_products(plan, store, w.params[:1])
    t1 = max(time.perf_counter() - t0, 1e-6)
    cores = max(1, min(32, len(os.sched_getaffinity(0))))
    n = int(max(1, min(w.n_templates, cores * budget_s / t1)))
    rows = w.params[np.sort(np.random.default_rng(seed).choice(w.n_templates, size=n, replace=False))]
    if n < 4 * cores:
        cores = 1
    if cores == 1:
        t0 = time.perf_counter()
        pairs = int((oin.inner_products(plan, store, rows)["kc"] >= 0).sum())
        return pairs / (time.perf_counter() - t0), n, time.perf_counter() - t0, pairs, 1
    blk = max(1, n // (4 * cores))
    # "spawn": this process holds a CUDA context, which must not be forked
    with mp.get_context("spawn").Pool(cores, initializer=_oracle_init,
                                      initargs=(dict(w.desc), w.bins, w.psd_scale, w.psd_shape, w.response)) as pool:
        pool.map(_oracle_rows, [rows[:1]] * cores)                       # workers up and warm before the clock starts
        t0 = time.perf_counter()
        pairs = sum(pool.map(_oracle_rows, [rows[i:i + blk] for i in range(0, n, blk)]))
        dt = time.perf_counter() - t0
    return pairs / dt, n, dt, pairs, cores


# ---------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""
    def __init__(self, index, period=0.002):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.period, self._stop, self._th = period, threading.Event(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {getattr(nv, k): v for k, v in (
            ("nvmlClocksEventReasonHwSlowdown", "hw_slowdown"),
            ("nvmlClocksThrottleReasonHwSlowdown", "hw_slowdown"),
            ("nvmlClocksThrottleReasonHwThermalSlowdown", "hw_thermal_slowdown"),
            ("nvmlClocksThrottleReasonSwThermalSlowdown", "sw_thermal_slowdown"),
            ("nvmlClocksThrottleReasonSwPowerCap", "sw_power_cap")) if hasattr(nv, k)}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.nv is not None:
            self._th = threading.Thread(target=self._run, daemon=True)
            self._th.start()

    def stop(self):
        self._stop.set()
        if self._th:
            self._th.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------
def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    w = make_workload(args.workload, 0, args.templates, args.n_sft, args.K)
    oin, plan, store = oracle_objects(w)
    # one step = a bounded sample: n_ref templates x all SFTs, sized from a probe so that the
    # whole run (steps + warmup) ends within a few minutes
    t0 = time.perf_counter()
    oin.inner_products(plan, store, w.params[:1])
    t1 = time.perf_counter() - t0
    total = args.steps + args.warmup
    n_ref = int(max(1, min(w.n_templates, 120.0 / total / max(t1, 1e-6), 64)))
    P = w.params[:n_ref]
    for _ in range(args.warmup):
        oin.inner_products(plan, store, P)
    pairs = 0
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r = oin.inner_products(plan, store, P)
        pairs += int((r["kc"] >= 0).sum())
    dt = time.perf_counter() - t0
    val = pairs / dt
    sample = "%d of %d templates x all %d SFT slots per step (oracle.inner.inner_products, numpy fp64)" % (
        n_ref, w.n_templates, w.desc["n_sft"])
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "templates_per_step": n_ref, "n_sft": w.desc["n_sft"], "K": w.desc["K"],
                   "kernel": w.desc["kernel"]},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores_used(), "kind": "oracle", "sample": sample,
                         "host_cores_available": len(os.sched_getaffinity(0))},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}), flush=True)


def aux_measurements(w2, plan, dev, stream, flush, pk, steps=5, warmup=3):
    """Beside the headline line: the two other calls of the library on the same data, a few steps each, so that the
    driver's record carries them - (i) ``sft_cumulative_snr`` on BASELINE.json configs[2] (16,384 templates, SNR(t) matrix
    16,384 x 10,800 fp32 = 708 MB written per step), (ii) ``sft_compute_sfts`` on a config-2 shaped
    series (HBM roofline).  Each carries its own roofline and clocks."""
    import torch
    from paper_2502_11823_b200 import api, workloads as wl
    out = {}
    w3 = wl.et_bns_bank(w2, 16384, bank_seed=6)                 # = workloads.config3(): same data, the 16,384-template bank
    w3.name = "config3-F"
    nT, N = w3.n_templates, plan.n_sft
    P = torch.from_numpy(np.ascontiguousarray(w3.params)).to(dev)
    ns = 64
    kc = torch.empty((ns, plan.n_channels, N), dtype=torch.int32, device=dev)
    x3 = [torch.empty(ns, dtype=torch.float64, device=dev) for _ in range(3)]
    plan.inner_products(P[:ns].contiguous(), x3[0], x3[1], x3[2], kc)
    plan.sync()
    pairs = int((kc >= 0).sum().item()) * nT // ns
    paths = plan.path_counts()
    snr = torch.empty((nT, N), dtype=torch.float32, device=dev)
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    ms, kms = 0.0, []
    for i in range(warmup + steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        plan.cumulative_snr(P, snr, None, None)
        b.record(stream)
        torch.cuda.synchronize()
        if i >= warmup:
            ms += a.elapsed_time(b)
            kms.append(plan.last_kernel_ms())
    clocks = sampler.stop()
    ms /= steps
    roof = roofline(w3, pairs, float(np.mean(kms)), paths, "auto", pk)
    hbm, src = hbm_peak()
    roof["output_hbm"] = {"bytes_written_per_step": int(snr.numel() * 4), "achieved_gbs": snr.numel() * 4 / (ms * 1e-3) / 1e9,
                          "peak_gbs": hbm, "peak_source": src}
    out["config3_cumulative_snr"] = {"value": pairs / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "steps": steps, "warmup": warmup,
                                     "templates": nT, "active_pairs": pairs, "gpu_launches_per_step": 2, "roofline": roof,
                                     "clocks": clocks}
    del snr, P, kc
    out["ingest_compute_sfts"] = ingest_measurement(steps=steps, warmup=warmup, dev=dev, stream=stream, flush=flush)
    return out


def hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ingest_measurement(steps, warmup, dev, stream, flush):
    """sft_compute_sfts on a series shaped like config 2 (10,800 segments of 16,384 float64 samples, 1.42 GB, device
    resident; band bins 5..186).  HBM-bound: the series is read once."""
    import torch
    from paper_2502_11823_b200 import api
    n_sft, n, k_lo, k_hi, dt = 10800, 16384, 5, 187, 1.0 / 2048.0
    g = torch.Generator(device=dev)
    g.manual_seed(11)
    x = torch.randn(n_sft * n, dtype=torch.float64, device=dev, generator=g) * 1e-23
    bins = torch.empty((n_sft, k_hi - k_lo), dtype=torch.complex64, device=dev)
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    ms = 0.0
    for i in range(warmup + steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        api.compute_sfts(x, n_sft, n, dt, k_lo, k_hi, bins, device=dev.index or 0, stream=stream.cuda_stream)
        b.record(stream)
        torch.cuda.synchronize()
        if i >= warmup:
            ms += a.elapsed_time(b)
    clocks = sampler.stop()
    ms /= steps
    nbytes = x.numel() * 8 + bins.numel() * 8
    peak, src = hbm_peak()
    gbs = nbytes / (ms * 1e-3) / 1e9
    return {"metric": "data-SFT generation (sft_compute_sfts)", "value": x.numel() / (ms * 1e-3), "unit": "samples/s",
            "ms_per_step": ms, "steps": steps, "warmup": warmup, "dtype": "f32 (f64 input)", "data": "synthetic",
            "config": {"workload": "config2-shaped series", "n_sft": n_sft, "n": n, "band": [k_lo, k_hi],
                       "cache": "l2_flush_between_steps; includes the end-of-call sync"},
            "clocks": clocks,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                         "traffic": None, "peak_source": src, "alg_bytes": nbytes}}


def aggregate_over_ranks(ms_dev, ms_host_step, pairs, device, world):
    """Whole-job numbers from per-rank ones: time = MAX over ranks (the slowest rank ends the step),
    work = SUM over ranks (each rank has its own template shard; no data-path collective)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_dev, ms_host_step, float(pairs)], dtype=torch.float64, device=device)
    if world > 1:
        tmax = t.clone()
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        tsum = t.clone()
        dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
        return float(tmax[0]), float(tmax[1]), float(tsum[2])
    return float(t[0]), float(t[1]), float(t[2])


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2502_11823_b200 import api, build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if local_rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    w = make_workload(args.workload, rank, args.templates, args.n_sft, args.K)
    stream = torch.cuda.current_stream()
    plan = api.plan_from_workload(w, device=local_rank, stream=stream.cuda_stream, evaluator=args.evaluator)
    if args.chunk:
        plan.set_chunk(args.chunk)
    nT = w.n_templates
    P_host = torch.from_numpy(np.ascontiguousarray(w.params)).pin_memory()
    P_dev = P_host.to(dev)
    xh = torch.empty(nT, dtype=torch.float64, device=dev)
    hh = torch.empty_like(xh)
    xi = torch.empty_like(xh)
    out_host = [torch.empty(nT, dtype=torch.float64).pin_memory() for _ in range(3)]
    out_np = [t.numpy() for t in out_host]
    P_np = P_host.numpy()
    # active pairs of this rank's bank, counted once by the library itself (k_c >= 0)
    kc = torch.empty((nT, plan.n_channels, plan.n_sft), dtype=torch.int32, device=dev)
    plan.inner_products(P_dev, xh, hh, xi, kc)
    plan.sync()
    pairs = int((kc >= 0).sum().item())
    paths = plan.path_counts()
    del kc
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    cumulative = args.workload == "config3"        # BASELINE.json configs[2]: the SNR(t) matrix is the output
    d2h_bytes = 3 * nT * 8
    if cumulative:
        snr_dev = torch.empty((nT, plan.n_sft), dtype=torch.float32, device=dev)
        snr_host = torch.empty((nT, plan.n_sft), dtype=torch.float32).pin_memory()
        snr_np = snr_host.numpy()
        d2h_bytes = int(snr_np.nbytes)

    def step_device():
        if cumulative:
            plan.cumulative_snr(P_dev, snr_dev, None, None)
        else:
            plan.inner_products(P_dev, xh, hh, xi, None)

    def step_host():
        if cumulative:
            plan.cumulative_snr(P_np, snr_np, None, None)
        else:
            plan.inner_products(P_np, out_np[0], out_np[1], out_np[2], None)

    def timed(fn, steps, warmup, record_kernel=False):
        for _ in range(warmup):
            flush.zero_()
            fn()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        kms = []
        l0 = plan.launch_count()
        for a, b in ev:
            flush.zero_()
            a.record(stream)
            fn()
            b.record(stream)
            if record_kernel:
                kms.append(plan.last_kernel_ms())
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        ms = sum(a.elapsed_time(b) for a, b in ev)
        return ms, plan.launch_count() - l0, kms

    sampler = ClockSampler(local_rank)
    sampler.start()
    ms_dev, launches, kms = timed(step_device, args.steps, args.warmup, record_kernel=True)
    clocks = sampler.stop()
    e2e_steps = max(3, min(args.steps, 5 if cumulative else 50))
    ms_host, _, _ = timed(step_host, e2e_steps, 3)
    ok = bool(torch.isfinite(xh).all().item() and (hh >= 0).all().item())
    ms_dev, ms_host_step, pairs_all = aggregate_over_ranks(ms_dev, ms_host / e2e_steps, pairs, dev, world)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    ms_step = ms_dev / args.steps
    value = pairs_all / (ms_step * 1e-3)
    e2e = pairs_all / (ms_host_step * 1e-3)
    k_ms = float(np.mean(kms)) if kms else None
    # pipe rates of this GPU (Gop/s) and the schedulers' sustained rate on the table kernel's instruction mix with
    # every stall removed (instructions/clock/scheduler): the ceiling for that mix, beside the nominal peak
    pk = api.measure_alu_peaks(local_rank)
    roof = roofline(w, pairs, k_ms, paths, args.evaluator, pk)
    aux = None
    if world == 1 and args.workload == "config2" and not args.no_aux and not args.templates and not args.n_sft:
        aux = aux_measurements(w, plan, dev, stream, flush, pk)
    cpu_val, cpu_n, cpu_dt, cpu_pairs, cpu_cores = time_oracle(w, budget_s=args.cpu_budget)
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "templates_per_gpu": nT, "n_sft_slots": int(w.desc["n_sft"]),
                   "n_channels": int(w.desc["n_channels"]), "K": int(w.desc["K"]), "kernel": w.desc["kernel"],
                   "pn1": int(w.desc["pn1"]), "evaluator": args.evaluator,
                   "arithmetic": "fp32 evaluators and contraction, fp64 phase/frequency track, fp64 accumulators",
                   "call": "sft_cumulative_snr" if cumulative else "sft_inner_products", "active_pairs_per_gpu": pairs, "bin_terms_per_gpu": pairs * (2 * w.desc["K"] + 1),
                   "parallelism": "templates sharded over %d GPU(s), data store replicated, no collective" % world,
                   "cache": "l2_flush_between_steps (256 MiB memset, outside the per-step events)"},
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": int(P_np.nbytes), "d2h_bytes_per_step": int(d2h_bytes),
                "ms_per_step": ms_host_step, "steps": e2e_steps},
        "gpu_launches": int(launches), "kernel_ms": k_ms, "results_finite": ok,
        "clocks": clocks, "roofline": roof, "aux": aux,
        "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cpu_cores, "kind": "oracle",
                         "host_cores_available": len(os.sched_getaffinity(0)),
                         "sample": "%d seeded templates (rng 99) of %d x all %d SFT slots (%d active pairs) in %.1f s, "
                                   "oracle.inner.inner_products numpy fp64, one worker process per core" % (
                                       cpu_n, nT, w.desc["n_sft"], cpu_pairs, cpu_dt)},
    }
    print(json.dumps(out), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()


# DRAM bytes (read + write) of one main-kernel launch, from the committed ncu --set full captures (dram__bytes_read.sum +
# dram__bytes_write.sum): NOT measured by this run - the source capture is named in roofline.traffic_source.
NCU_TRAFFIC = {
    ("config2-F", "auto"): (2.103808e6 + 75.008e3, "profiles/r02_main_kernel.md"),
    ("config2-F", "table"): (2.103808e6 + 75.008e3, "profiles/r02_main_kernel.md"),
    ("config2-F", "direct"): (8.213504e6 + 10.752e3, "profiles/r01d_kernel_v7_tables.md"),
    ("config3-F", "auto"): (38.722304e6 + 831.203584e6, "profiles/r02_main_kernel.md"),
    ("config4", "auto"): (6.319616e6 + 229.888e3, "profiles/r02_main_kernel.md"),
}

# Algorithmic work per active pair and the ALU peak: DESIGN.md section 7.
SM_COUNT, SM_MAX_GHZ = 148, 1.965
S_ORDER = {"series0": 1, "series1": 4, "series2": 11, "series3": 16}     # packed-lane ops of the far-bin recurrence


def alg_instr_per_pair(path, K, C):
    """The FIXED per-unit figure of the roofline: warp instructions of the moment-table / series /
    closed-Fresnel formulation per active (template, SFT) pair on evaluator path ``path``, as counted for the round-1 kernel
    (closed-form fp64 track 50 + SFT loop 13 + phase/prefactor/response/accumulation 23 (+12 per extra channel); table tier 1:
    21 + 38 per channel, tier 2: 21 + 134 per channel; series order n: per far bin 2.5 + s_n/2 + 1 + 3.5 C, central bin
    7(n+1) + 2 + 7 C; closed Fresnel form: 64 + 3.5 C per bin; a packed FFMA2/FMUL2 = ONE instruction).  It is kept fixed so
    that fractions stay comparable from round to round: a kernel that needs fewer instructions for the same pairs (the
    polynomial track of round 2) shows up as a higher fraction, exactly as a faster kernel should."""
    fixed = 86 + 12 * (C - 1)
    if path == "table":
        return fixed + 21 + 38 * C
    if path == "table2":                 # 14 loads, 71 packed FMAs + 22 scalings for S1, 24 + 3 for H
        return fixed + 21 + 134 * C
    if path == "fresnel":
        return fixed + (2 * K + 1) * (64 + 3.5 * C)
    n = int(path[-1])
    return fixed + 2 * K * (2.5 + S_ORDER[path] / 2.0 + 1 + 3.5 * C) + 7 * (n + 1) + 2 + 7 * C


def kernel_instr_per_pair(path, K, C, strict=False):
    """What the CURRENT kernel issues per pair on its common path (clean block, polynomial track, tier-1 tables; counted
    in the SASS of the hot loop, profiles/r02_main_kernel.md: 225 instructions per two SFTs): track 29 (11 fp64, 3
    conversions, 13 fp32, 2 constant loads), S1 29 C (19 packed FMAs + 10 scalings), H 4 C (compact node), 5 C table loads,
    prefactor 15 + 12 (C - 1), accumulation 3; plus - not in the strict count - node / address arithmetic 18 C and the loop
    over the presence mask 9.5.  Other paths as in alg_instr_per_pair."""
    if path == "table":
        core = 29 + (29 + 4 + 5) * C + 15 + 12 * (C - 1) + 3
        return core if strict else core + 18 * C + 9.5
    full = alg_instr_per_pair(path, K, C)
    return full - 34 if strict else full           # strict: without the 13 loop + 21 node/constant instructions


def roofline(w, pairs, kernel_ms, paths, evaluator="auto", pk=None):
    """Issue-slot roofline of the fused main kernel.  The data are L2/L1 resident, so the path is
    bound by plain ALU work; no single pipe dominates (ncu: FMA 34 %, XU 31 %, LSU 22 %, ALU 17 %, FP64 15 %) and the
    binding resource is the warp schedulers' issue rate: peak = 148 SMs x 4 schedulers x 1 warp instruction/clock x 32 lanes
    x 1.965 GHz (numerically the FP32 lane peak).  achieved = per-pair figure of the measured path mix x 32 lanes x
    warp-pairs / kernel time (CUDA events around the launch on the plan's stream)."""
    if not kernel_ms or not paths:
        return None
    K, C = int(w.desc["K"]), int(w.desc["n_channels"])
    tot = float(sum(paths.values()))
    mix = {k: v / tot for k, v in paths.items() if v}
    peak = SM_COUNT * 4 * 32 * SM_MAX_GHZ          # G lane-instructions/s
    rate = (pairs / C) / (kernel_ms * 1e-3) / 1e9  # G (template, SFT) lane-pairs/s; pairs counts channels, tracks do not

    def per_pair(fn, **kw):
        return sum(f * fn(k, K, C, **kw) for k, f in mix.items())

    ops_fixed = per_pair(alg_instr_per_pair)
    ops_kernel = per_pair(kernel_instr_per_pair)
    ops_strict = per_pair(kernel_instr_per_pair, strict=True)
    traffic, tsrc = NCU_TRAFFIC.get((w.name, evaluator), (None, None))
    r = {"bound": "alu", "achieved": ops_fixed * rate, "peak": peak, "unit": "G lane-instructions/s (issue slots)",
         "frac": ops_fixed * rate / peak, "traffic": traffic,
         "traffic_source": ("ncu capture " + tsrc + " (not measured by this run)") if tsrc else None,
         "kernel": "sft_main_kernel", "kernel_ms": kernel_ms,
         "alg_instr_per_pair": ops_fixed,
         "alg_instr_source": "fixed per-unit figure of DESIGN.md section 7 (formulation as counted in round 1)",
         "alg_instr_strict_fixed": ops_fixed - 34.0, "frac_strict_fixed": (ops_fixed - 34.0) * rate / peak,   # fixed count without its 13 loop + 21 node/constant instructions
         "kernel_instr_per_pair": ops_kernel, "frac_kernel_count": ops_kernel * rate / peak,
         "alg_instr_strict": ops_strict, "frac_strict": ops_strict * rate / peak,
         "path_mix": mix,
         "peak_source": "nominal: 148 SM x 4 schedulers x 32 lanes x 1.965 GHz (B200_PROFILING.md unit counts/clocks), DESIGN.md section 7"}
    if pk:
        # against what this GPU measurably issues: plain FFMA lane rate (one instruction per clock and scheduler in practice)
        # and the ceiling of the table kernel's own instruction mix with every stall removed
        r["measured_alu"] = pk
        if pk.get("ffma"):
            r["frac_of_measured_ffma_issue"] = ops_fixed * rate / pk["ffma"]
        if pk.get("table_mix_ipc"):
            r["frac_of_mix_ceiling"] = r["frac"] / pk["table_mix_ipc"]
    return r


def run_sweep(args):
    """--sweep: BASELINE.json configs[4], one axis at a time around the config-2 point (templates,
    SFTs, band half-width K, evaluator).  One JSON line per point: throughput, main-kernel time,
    issue-slot roofline fraction and the normalised error against the oracle on 3 sampled templates.
    The phase-path axis (fp64 vs split-fp32 = double-float track) is run at the config-2 point for both
    evaluators."""
    import torch
    from paper_2502_11823_b200 import api, build, workloads as wl
    from oracle import inner as oin
    build.build()
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    points = []
    for nt in [4 ** i for i in range(0, 11)]:
        points.append(dict(axis="templates", n_templates=nt, n_sft=10800, K=8, evaluator="auto"))
    for ns in (1024, 2700, 10800, 43200):
        points.append(dict(axis="n_sft", n_templates=4096, n_sft=ns, K=8, evaluator="auto"))
    for K in (2, 4, 8, 16, 32, 64):
        for ev in ("auto", "direct"):
            points.append(dict(axis="K", n_templates=4096, n_sft=10800, K=K, evaluator=ev))
    for ph in ("fp64", "split32"):
        for ev in ("auto", "direct"):
            points.append(dict(axis="phase_path", n_templates=4096, n_sft=10800, K=8, evaluator=ev, phase_path=ph))
    cache = {}
    for pt in points:
        key = (pt["n_sft"], pt["K"])
        if key not in cache:
            cache.clear()
            cache[key] = wl.et_bns(n_templates=4096, n_sft=pt["n_sft"], K=pt["K"], name="config5")
        w0 = cache[key]
        nT = pt["n_templates"]
        w = wl.et_bns_bank(w0, nT) if nT != 4096 else w0
        plan = api.plan_from_workload(w, device=0, stream=stream.cuda_stream, evaluator=pt["evaluator"],
                                      phase_path=pt.get("phase_path", "fp64"))
        P = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
        xh = torch.empty(nT, dtype=torch.float64, device=dev)
        hh, xi = torch.empty_like(xh), torch.empty_like(xh)
        ns = min(nT, 64)                                        # active pairs and path mix from a sample
        kc = torch.empty((ns, 1, plan.n_sft), dtype=torch.int32, device=dev)
        plan.inner_products(P[:ns].contiguous(), xh[:ns], hh[:ns], xi[:ns], kc)
        plan.sync()
        pairs = int((kc >= 0).sum().item()) * nT // ns
        paths = plan.path_counts()
        steps = 20 if nT <= 65536 else 5
        kms, ms = [], 0.0
        for i in range(3 + steps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            plan.inner_products(P, xh, hh, xi, None)
            b.record(stream)
            torch.cuda.synchronize()
            if i >= 3:
                ms += a.elapsed_time(b)
                kms.append(plan.last_kernel_ms())
        rows = np.unique([0, nT // 2, nT - 1])
        op, st = oracle_objects(w)[1:]
        o = oin.inner_products(op, st, w.params[rows])
        norm = np.sqrt(oin.xx_band(op, st) * o["hh"])
        g_xh, g_hh = xh.cpu().numpy()[rows], hh.cpu().numpy()[rows]
        err = float(max(np.max(np.abs(g_xh - o["xh"]) / norm), np.max(np.abs(g_hh - o["hh"]) / norm)))
        roof = roofline(w, pairs, float(np.mean(kms)), paths, pt["evaluator"])
        print(json.dumps(dict(pt, workload="config5", active_pairs=pairs, ms_per_step=ms / steps,
                              kernel_ms=float(np.mean(kms)), pairs_per_s=pairs / (ms / steps * 1e-3),
                              roofline_frac=roof["frac"], alg_instr_per_pair=roof["alg_instr_per_pair"],
                              path_mix=roof["path_mix"], oracle_err=err, phase_path=pt.get("phase_path", "fp64"))), flush=True)
        plan.close()
        del P, xh, hh, xi, kc


def run_ingest(args):
    """--ingest: SURVEY section 8(f) NEXT-1 - one JSON line: samples/s and achieved GB/s against the measured copy bandwidth."""
    import torch
    from paper_2502_11823_b200 import build
    build.build()
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    print(json.dumps(ingest_measurement(args.steps, args.warmup, dev, torch.cuda.current_stream(), flush)), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2")
    ap.add_argument("--templates", type=int, default=None)
    ap.add_argument("--n-sft", type=int, default=None, dest="n_sft")
    ap.add_argument("--K", type=int, default=None)
    ap.add_argument("--chunk", type=int, default=0)
    ap.add_argument("--evaluator", default="auto", choices=["auto", "direct", "table"])
    ap.add_argument("--sweep", action="store_true", help="config-5 scaling sweep (one JSON line per point)")
    ap.add_argument("--ingest", action="store_true", help="time the GPU data-SFT generation (NEXT-1)")
    ap.add_argument("--cpu-budget", type=float, default=12.0, dest="cpu_budget")
    ap.add_argument("--no-aux", action="store_true", dest="no_aux", help="skip the config-3 and ingest side measurements")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.sweep or args.ingest:
        if rank == 0:
            run_sweep(args) if args.sweep else run_ingest(args)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
