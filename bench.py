#!/usr/bin/env python
"""bench.py -- SPIIR template-bank filter throughput on B200 (BASELINE.json metric and config).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

One "step" = one pass of the whole hot path over one batch of synthetic input: the streaming run of
BASELINE.json:configs[3] (4096 templates x 1024 filters, 262 144 float32 samples fed as 16 chunks of 16 384
with state carry), i.e. 16 spiir_filter calls = 1.0995e12 filter-samples.  Inputs are resident in HBM when the
timed region starts (`value`); `e2e` repeats the measurement through spiir_filter_host_async / spiir_bank_host_sync with host buffers
(H2D of every chunk and D2H of every SNR block inside the timed region).  Prints ONE JSON line.

The default run (N = 1, --config 3) also times every other config of BASELINE.json in short legs and reports them
under `per_config` (cfg0, cfg1 one-shot and 16 x 4096, cfg2, cfg4, two banks of small templates: filter-samples/s, roofline fraction, per-call
p50/p99, path taken, clocks of that leg); --no-per-config skips them.

N > 1 (torchrun, one rank per GPU): templates are independent, so every rank filters
its own seeded 4096-template bank -- no data-path collective -- and `value` is the total over ranks divided by
the slowest rank's time ("scaling": "weak").  With --shard ONE bank is split over the ranks by template
(shard_templates, longest-processing-time bin packing; "scaling": "strong"; per-rank filter counts in `shard`).

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores, on a bounded sample of the
same workload; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import spiir_inputs  # noqa: E402

METRIC = "SPIIR filter-samples/s (templates x filters x samples)"
UNIT = "filter-samples/s"
FLOPS_PER_FILTER_SAMPLE = 12          # complex*complex 6 + real*complex 2 + complex add 2 + sum 2
N_SM, LANES, BOOST_HZ = 148, 128, 1.965e9   # B200: SMs x FP32 lanes x 2 flops x clocks.max.sm (MEASURED_PEAKS.json sm_max_mhz)
FP32_PEAK_TFLOPS = N_SM * LANES * 2 * BOOST_HZ / 1e12    # 74.4 TFLOP/s, derivation in DESIGN.md section 7
# dram__bytes_read.sum + dram__bytes_write.sum of one spiir_filter_kernel launch (cfg3, default blocking, 8192 samples)
# from the committed ncu --set full capture profiles/r02_filter_kernel_full.md: 119.3 MB + 244.6 MB
NCU_TRAFFIC_CFG3_LAUNCH = 363.8e6
# the same for one spiir_stream_kernel launch of cfg4 (16 samples), profiles/r02_cfg4_stream_launches.md: 144.6 MB + 18.2 MB
NCU_TRAFFIC_CFG4_LAUNCH = 162.8e6


def measured_hbm_peak():
    """(GB/s, source): the driver-measured copy bandwidth of this pool's B200s, else the profiling guide's fallback."""
    try:
        d = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)"


def workload_name(inp):
    return (f"{inp.name}: {inp.n_templates} templates x {inp.n_filters // max(inp.n_templates, 1)} filters (mean), "
            f"{inp.n_samples} samples, streaming in {inp.chunk}-sample chunks")


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML; nvidia-smi semantics)."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _loop(self):
        nv = self._nv
        names = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "sw_power_cap": 0x4, "hw_power_brake_slowdown": 0x80}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.05)

    def __enter__(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def time_oracle(inp, n_templates: int, n_threads: int = 0):
    """CPU oracle on the first n_templates templates of inp, all samples, streaming in inp.chunk chunks."""
    import oracle
    sub = inp.select_templates(np.arange(min(n_templates, inp.n_templates)))
    oracle.build()
    st = oracle.Stream(sub.offsets, sub.a1, sub.b0, sub.delays)
    t0 = time.perf_counter()
    for c0 in range(0, sub.n_samples, sub.chunk):
        st.filter(sub.x[c0:c0 + sub.chunk], n_threads)
    dt = time.perf_counter() - t0
    st.close()
    return sub.filter_samples / dt, dt, sub, oracle.max_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    inp = spiir_inputs.make_config(args.config)
    n_tpl = args.ref_templates
    for _ in range(args.warmup):
        time_oracle(inp, max(1, n_tpl // 8))
    rates, times = [], []
    for _ in range(args.steps):
        r, dt, sub, cores = time_oracle(inp, n_tpl)
        rates.append(r)
        times.append(dt)
    total_fs = sub.filter_samples * args.steps
    value = total_fs / sum(times)
    sample = f"first {sub.n_templates} of {inp.n_templates} templates, all {inp.n_samples} samples, {inp.chunk}-sample chunks"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(inp), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def setup(args):
    """Device, process group and library for this rank -> (torch, dist, pkg, world, rank, dev_index, red_dev, oversubscribed)."""
    import torch
    import torch.distributed as dist
    import paper_1602_05573_b200 as pkg

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the SPIIR library has no CPU fallback")
    n_dev = torch.cuda.device_count()
    # fewer GPUs than ranks (or SPIIR_BENCH_BACKEND=gloo): a functional check of the multi-rank path only -- NCCL cannot put
    # two ranks on one GPU, so the timing exchange then goes over gloo on the host and the line says "functional_only"
    oversubscribed = world > 1 and (world > n_dev or os.environ.get("SPIIR_BENCH_BACKEND") == "gloo")
    dev_index = local_rank % n_dev
    torch.cuda.set_device(dev_index)
    red_dev = "cpu" if oversubscribed else "cuda"
    if world > 1:
        if oversubscribed:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", dev_index))
    if not pkg.library_path().exists():
        # the in-tree library normally travels with the repo; build it once (local rank 0) if it does not
        if local_rank == 0:
            from paper_1602_05573_b200.build import build as build_cuda
            build_cuda()
        else:
            t_wait = time.time()
            while not pkg.library_path().exists() and time.time() - t_wait < 600:
                time.sleep(1.0)
    pkg.load_library()
    return torch, dist, pkg, world, rank, dev_index, red_dev, oversubscribed


def measure(ctx, args, cfg, steps, warmup, *, chunk=None, e2e=False, label=None, inp=None):
    """Time `steps` steps of configs[cfg] on this rank's GPU (a step = the config's whole streaming run; chunk=0: one call
    over the whole series).  -> dict with value, ms_per_step, roofline, latency, clocks, launches, path (+ e2e)."""
    torch, dist, pkg, world, rank, dev_index, red_dev, oversubscribed = ctx
    inp = spiir_inputs.make_config(cfg) if inp is None else inp        # inp given: a workload outside BASELINE.json:configs
    shard_info = None
    if args.shard and world > 1:
        # ONE bank split over the ranks by template: longest-processing-time
        # bin packing on the filter counts, no data-path collective, every rank filters the same strain
        parts = pkg.shard_templates(inp.offsets, world)
        kt = np.diff(inp.offsets)
        loads = [int(kt[p_].sum()) for p_ in parts]
        shard_info = {"filters_per_rank": loads, "templates_per_rank": [int(p_.size) for p_ in parts],
                      "imbalance_max_over_mean": max(loads) / (sum(loads) / world)}
        total_filters = inp.n_filters
        inp = inp.select_templates(parts[rank])
    elif rank > 0:
        # weak scaling: every rank filters its own seeded bank of the config's size (same distributions, another bank)
        rng = np.random.default_rng(spiir_inputs.SEED0 + 1000 * rank + cfg)
        inp = inp.select_templates(rng.permutation(inp.n_templates))
    N, T = inp.n_samples, inp.n_templates
    L = inp.chunk if chunk is None else (N if chunk == 0 else chunk)
    path = args.path
    if path == 0 and L <= 64 and inp.n_filters >= (1 << 20):
        path = pkg.PATH_STREAM            # tiny chunks over a large bank: the HBM-bound streaming blocking
    opt = pkg.SpiirOptions(path=path, filters_per_thread=args.filters_per_thread, warps_per_cta=args.warps_per_cta,
                           window_copies=args.window_copies, scan_segments=args.scan_segments,
                           scan_launches=args.scan_launches)
    bank = pkg.SpiirBank(inp.offsets, inp.a1, inp.b0, inp.delays, dev_index, opt)
    x = torch.from_numpy(inp.x).cuda()
    keep_whole = (T * N * 8) <= args.max_snr_bytes
    snr = torch.empty((T, N if keep_whole else L), dtype=torch.complex64, device="cuda")
    stream = torch.cuda.current_stream()
    peak_power = torch.empty(T, dtype=torch.float32, device="cuda")
    peak_index = torch.empty(T, dtype=torch.int32, device="cuda")
    n_calls = (N + L - 1) // L

    # the tensor views of every call are made once (slicing a tensor costs more host time than a cfg0 call takes on the GPU)
    views, calls = [], []
    for c0 in range(0, N, L):
        n = min(L, N - c0)
        views.append((x[c0:c0 + n], snr[:, c0:c0 + n] if keep_whole else snr[:, :n]))
        calls.append(pkg.spiir_filter_prepared(bank.handle, views[-1][0], views[-1][1], stream=stream))

    def one_step(events=None):
        bank.reset()
        for i, (xin, out) in enumerate(views):
            if events is not None:
                events[i].record(stream)
            if args.peaks:
                pkg.spiir_filter_peaks(bank.handle, xin, peak_power, peak_index, None if args.peaks == 1 else out)
            else:
                calls[i]()                  # = pkg.spiir_filter(bank.handle, xin, out), arguments marshalled once
        if events is not None:
            events[n_calls].record(stream)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(warmup, 3)):
        one_step()
    barrier()
    launches0 = pkg.spiir_kernel_launches()
    start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(dev_index) as clocks:
        barrier()
        start.record(stream)
        for s in range(steps):
            one_step()                      # the timed region carries no per-call events: they would sit between the
        stop.record(stream)                 # kernels of consecutive calls and break their programmatic launch chain
        barrier()
    launches = pkg.spiir_kernel_launches() - launches0
    elapsed_ms = start.elapsed_time(stop)
    # per-call latency: a separate pass with one event pair per call (at most 2 steps' worth of calls)
    lat_steps = min(steps, 2 if n_calls > 64 else 50)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(n_calls + 1)] for _ in range(lat_steps)]
    for s in range(lat_steps):
        one_step(ev[s])
    barrier()
    call_ms = [ev[s][i].elapsed_time(ev[s][i + 1]) for s in range(lat_steps) for i in range(n_calls)]
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=red_dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    elapsed_ms_max = float(t.item())
    fs_step = inp.filter_samples
    if shard_info is not None:
        value = total_filters * N * steps / (elapsed_ms_max * 1e-3)      # one bank over all ranks: strong scaling
        shard_info["rank0_ms_per_step"] = elapsed_ms / steps
    else:
        value = world * fs_step * steps / (elapsed_ms_max * 1e-3)

    # dominant kernel: spiir_filter_kernel (1 or 2 launches per spiir_filter call; the call also enqueues one device-to-
    # device append of the chunk, < 0.1 % of the call)
    fs_call = inp.n_filters * L
    avg_call_s = elapsed_ms * 1e-3 / (steps * n_calls)      # timed region (includes the reset of each step)
    achieved_tflops = FLOPS_PER_FILTER_SAMPLE * fs_call / avg_call_s / 1e12
    launches_per_call = max(1.0, launches / float(steps * n_calls))      # kernel launches of one spiir_filter call
    traffic = args.ncu_traffic_bytes
    default_blocking = not (args.filters_per_thread or args.warps_per_cta or args.window_copies or args.path)
    if traffic is None and cfg == 3 and default_blocking and chunk is None:
        traffic = NCU_TRAFFIC_CFG3_LAUNCH
    if traffic is None and cfg == 4 and not (args.filters_per_thread or args.warps_per_cta or args.window_copies) and chunk is None:
        traffic = NCU_TRAFFIC_CFG4_LAUNCH
    roofline = {"bound": "alu", "achieved": achieved_tflops, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                "frac": achieved_tflops / FP32_PEAK_TFLOPS, "traffic": traffic,
                "kernel": "spiir_filter_kernel", "launch_ms": avg_call_s * 1e3 / launches_per_call,
                "launches_per_call": launches_per_call, "call_ms": avg_call_s * 1e3,
                "algorithmic_flop_per_launch": FLOPS_PER_FILTER_SAMPLE * fs_call / launches_per_call,
                "algorithmic_hbm_bytes_per_launch": (8.0 * T * L + 36.0 * inp.n_filters * launches_per_call) / launches_per_call,
                "peak_source": "148 SMs x 128 FP32 lanes x 2 flop x 1965 MHz (clocks.max.sm); no driver-measured FP32 peak exists",
                "issue_slot_util": 8 * fs_call / avg_call_s / (N_SM * LANES * BOOST_HZ),
                "hbm_write_gbs": 8.0 * T * L / avg_call_s / 1e9}

    call_us = np.sort(np.asarray(call_ms)) * 1e3
    latency = {"calls": int(call_us.size), "samples_per_call": int(L), "p50_us": float(np.percentile(call_us, 50)),
               "p99_us": float(np.percentile(call_us, 99)), "max_us": float(call_us[-1]),
               "real_time_us_per_call": 1e6 * L / spiir_inputs.FS}
    if L <= 64:
        # tiny chunks: every call streams the whole bank through the SMs once -> HBM roofline
        bytes_call = inp.n_filters * 36.0 + 8.0 * T * L + 4.0 * L     # 20 B coefficients + 8 B state in + 8 B state out per filter
        peak_gbs, peak_src = measured_hbm_peak()
        roofline = {"bound": "hbm", "achieved": bytes_call / avg_call_s / 1e9, "peak": peak_gbs, "unit": "GB/s",
                    "frac": bytes_call / avg_call_s / 1e9 / peak_gbs, "traffic": traffic,
                    "kernel": "spiir_stream_kernel", "launch_ms": avg_call_s * 1e3 / launches_per_call,
                    "launches_per_call": launches_per_call, "call_ms": avg_call_s * 1e3, "peak_source": peak_src,
                    "algorithmic_bytes_per_call": bytes_call}

    res = {"workload": (label or workload_name(inp)) if chunk is None else f"{inp.name}: {T} templates, {N} samples, {n_calls} call(s) of {L}",
           "value": value, "unit": UNIT, "steps": steps, "ms_per_step": elapsed_ms_max / steps, "path": bank.last_path,
           "pct_of_fp32_fma_peak": 100.0 * FLOPS_PER_FILTER_SAMPLE * (value / world) / (FP32_PEAK_TFLOPS * 1e12),
           "gpu_launches": int(launches), "roofline": roofline, "latency": latency, "clocks": clocks.summary(),
           "snr_buffer": "whole [T][N]" if keep_whole else "per-chunk [T][L] reused",
           "l2": "each step writes %.2f GB of SNR and reads a %.0f MB bank" % (T * N * 8 / 1e9, inp.n_filters * 28 / 1e6),
           "_inp": inp}
    if shard_info is not None:
        res["shard"] = shard_info

    # ---- end to end through the public host-buffer entry (H2D + kernels + D2H inside the timed region)
    if e2e:
        xh = torch.from_numpy(inp.x).pin_memory()
        outh = torch.empty((2, T, L), dtype=torch.complex64).pin_memory()      # results land here, two chunks deep
        xh_np, outh_np = xh.numpy(), outh.numpy()

        def e2e_step():
            bank.reset()
            for i, c0 in enumerate(range(0, N, L)):
                n = min(L, N - c0)
                # enqueue H2D of the chunk, the kernels and the D2H of SNR[:, chunk]; the copies of chunk i overlap
                # the kernels of chunk i+1
                pkg.spiir_filter_host_async(bank.handle, xh_np[c0:c0 + n], outh_np[i & 1, :, :n])
            pkg.spiir_bank_host_sync(bank.handle)                               # every result of the step is in host memory

        e2e_step()
        barrier()
        e2e_steps = max(1, min(steps, args.e2e_steps))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        tt = torch.tensor([dt], dtype=torch.float64, device=red_dev)
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        fs_total = (total_filters * N) if shard_info is not None else world * fs_step
        res["e2e"] = {"value": fs_total * e2e_steps / float(tt.item()), "unit": UNIT,
                      "h2d_bytes_per_step": int(N * 4), "d2h_bytes_per_step": int(T * N * 8),
                      "steps": e2e_steps, "api": "spiir_filter_host_async per chunk + spiir_bank_host_sync per step (pinned host buffers)"}
        if keep_whole and not args.peaks:
            # the last chunk's host block must equal the device-resident run of the same chunking bit for bit
            c0 = (n_calls - 1) * L
            n = N - c0
            dev_last = snr[:, c0:c0 + n].cpu().numpy()
            res["e2e"]["last_chunk_bitwise_equal_to_device_run"] = bool(
                np.array_equal(outh_np[(n_calls - 1) & 1, :, :n].view(np.float32), dev_last.view(np.float32)))
    bank.close()
    del snr, x
    torch.cuda.empty_cache()
    return res


def run_ours(args):
    ctx = setup(args)
    torch, dist, pkg, world, rank, dev_index, red_dev, oversubscribed = ctx
    main = measure(ctx, args, args.config, args.steps, args.warmup, e2e=not args.no_e2e)
    inp = main.pop("_inp")
    line = {"metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": main["ms_per_step"], "higher_is_better": True,
            "scaling": "strong" if (args.shard and world > 1) else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": main["workload"], "path": main["path"],
                       "l2": main["l2"] + ": working set larger than the 126 MB L2", "snr_buffer": main["snr_buffer"],
                       "entry": ["spiir_filter", "spiir_filter_peaks (no SNR output)", "spiir_filter_peaks (+ SNR output)"][args.peaks]},
            "pct_of_fp32_fma_peak": main["pct_of_fp32_fma_peak"],
            "gpu_launches": main["gpu_launches"], "roofline": main["roofline"], "latency": main["latency"],
            "clocks": main["clocks"]}
    if "e2e" in main:
        line["e2e"] = main["e2e"]
    if "shard" in main:
        line["shard"] = main["shard"]
    if oversubscribed:
        line["functional_only"] = True          # ranks share a GPU: the value is not a multi-GPU number
        line["oversubscribed"] = True

    # ---- every other config of BASELINE.json, driver-timed in the same run (N = 1 only; short legs)
    if world == 1 and not args.no_per_config and args.config == 3:
        per = {}
        legs = [("cfg0", 0, None, 200), ("cfg1_oneshot", 1, 0, 20), ("cfg1_chunked", 1, None, 10), ("cfg2", 2, None, 5),
                ("cfg4", 4, None, 2)]
        # + banks of small templates: 37 888 templates of 32 filters and 75 776
        #   of 8 (two full waves of CTA items on 148 SMs each), cfg1's distributions, delays up to 2047, 4 calls of 4096 samples
        small = {"small_templates_32": (32, 37888), "small_templates_8": (8, 75776)}
        legs += [(name, -1, None, 5) for name in small]
        for name, cfg, chunk, steps in legs:
            override = None
            if name in small:
                kt, nt = small[name]
                override = spiir_inputs.make_random_bank(7 + kt, [kt] * nt, 16384, d_max=2047, chunk=4096, name=name)
            r = measure(ctx, args, cfg, steps, 3, chunk=chunk, inp=override)
            r.pop("_inp")
            rf = r["roofline"]
            per[name] = {"workload": r["workload"], "value": r["value"], "unit": UNIT, "steps": steps, "ms_per_step": r["ms_per_step"],
                         "path": r["path"], "bound": rf["bound"], "achieved": rf["achieved"], "peak": rf["peak"],
                         "roofline_unit": rf["unit"], "frac": rf["frac"], "launches_per_call": rf["launches_per_call"],
                         "p50_us": r["latency"]["p50_us"], "p99_us": r["latency"]["p99_us"],
                         "call_us_back_to_back": rf["call_ms"] * 1e3, "samples_per_call": r["latency"]["samples_per_call"],
                         "clocks": r["clocks"]}
        line["per_config"] = per

    # ---- the CPU oracle beside it (rank 0, N = 1 only): a reported baseline, not the target
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        r, dt, sub, cores = time_oracle(inp, args.cpu_templates)
        line["cpu_baseline"] = {"value": r, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
                                "sample": f"first {sub.n_templates} of {inp.n_templates} templates, all {inp.n_samples} samples, {inp.chunk}-sample chunks"}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="index into BASELINE.json:configs (3 = headline)")
    ap.add_argument("--path", type=int, default=0, help="SPIIR_PATH_* override (0 auto)")
    ap.add_argument("--filters-per-thread", type=int, default=0)
    ap.add_argument("--warps-per-cta", type=int, default=0)
    ap.add_argument("--window-copies", type=int, default=0)
    ap.add_argument("--scan-segments", type=int, default=0)
    ap.add_argument("--scan-launches", type=int, default=0, help="3: three-launch form of the time-parallel path")
    ap.add_argument("--peaks", type=int, default=0, help="1: spiir_filter_peaks without SNR output, 2: with (not the headline)")
    ap.add_argument("--max-snr-bytes", type=float, default=20e9, help="keep the whole [T][N] SNR if it fits")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config legs (cfg0, cfg1, cfg2, cfg4) of the default run")
    ap.add_argument("--shard", action="store_true", help="N > 1: split ONE bank over the ranks by template (strong scaling)")
    ap.add_argument("--cpu-templates", type=int, default=96, help="templates of the bounded oracle sample")
    ap.add_argument("--ref-templates", type=int, default=32, help="templates per step of --impl reference")
    ap.add_argument("--ncu-traffic-bytes", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
