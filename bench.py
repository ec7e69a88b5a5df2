#!/usr/bin/env python
"""bench.py -- templates/s matched-filtered at N = 2^20 on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg1|cfg2|cfg3] [--impl ours|reference]

One "step" = one pass of the whole hot path (set_psd,
load_segment, template setup, SPA generation, correlate, inverse FFT, |z|/sigma, peak +
threshold, results) of ONE data segment against ONE bank, through the C ABI of
include/cbmf.h.  Default workload: BASELINE.json configs[1] (N = 2^20, fs = 4096 Hz,
1024 templates U[1,3]^2 Msun, 4 injections, threshold 6).

  value     templates/s, inputs and outputs resident in HBM (cbmf_*_dev entry points),
            CUDA events on the context's stream, L2 flushed between timed steps.
  e2e       the same step through the host-pointer entry points: pinned host PSD /
            samples / bank in, peaks and triggers out, every copy inside the timed region.
  roofline  dominant kernel (the slower of the two FFT passes): algorithmic flops per
            launch / mean launch duration (CUDA events around every launch of the pass,
            taken in a second set of K steps so the events do not perturb `value`).
  cpu_baseline  the CPU oracle (oracle/, fp64, as it stands) on a bounded sample of the
            same workload, host cores of this box.

Multi-GPU (torchrun, one rank per GPU): the bank is sharded by contiguous slices, the
segment is replicated, no data-path collective; weak scaling: every rank
filters a full-size bank slice.  --impl reference times the oracle (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "templates/sec matched-filtered at N=2^20 (1 B200) and % of FFT roofline"
UNIT = "templates/s"
# FP32 ALU peak of one B200 from unit counts and clocks (B200_PROFILING.md table: 148 SMs,
# clocks.max.sm 1965 MHz; 128 FP32 lanes per SM, FMA = 2 flop): DESIGN.md §6.
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def make_workload(name: str, world: int, rank: int):
    """Seeded synthetic workload; for world > 1 the bank is world x the config's size and
    this rank takes slice `rank` (weak scaling)."""
    from testsupport import workloads as W
    from paper_1006_4644_b200.sharding import shard_range
    wl = W.by_name(name)
    per_rank = wl.n_templates
    if world > 1:
        seed, lo, hi = {"cfg1": (3, 1.0, 3.0), "cfg2": (4, 1.0, 10.0), "cfg3": (5, 1.0, 5.0)}[name]
        full = W.draw_bank(seed, per_rank * world, lo, hi)      # first per_rank rows == the config's bank
        a, b = shard_range(per_rank * world, rank, world)
        wl.bank = np.ascontiguousarray(full[a:b])
    return wl


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""

    def __init__(self, index: int, period_s: float = 0.004):
        self.index, self.period = index, period_s
        self.sm, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self._nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nvml = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = index
            if vis:
                ids = [v for v in vis.split(",") if v.strip() != ""]
                if index < len(ids) and ids[index].strip().isdigit():
                    phys = int(ids[index])
            self._h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nvml = None

    def _run(self):
        n = self._nvml
        names = {
            "hw_slowdown": getattr(n, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(n, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(n, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(n, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(n, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.sm.append(float(n.nvmlDeviceGetClockInfo(self._h, n.NVML_CLOCK_SM)))
                r = int(n.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self._nvml is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                    "note": "nvml unavailable or region shorter than one sample"}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.sm)}


def pass_flops(n: int, lg1: int, lg2: int, n_b_mean: float):
    """Algorithmic flops per template of the two FFT passes:
    pass 1 = N1-point column FFTs (5 N log2 N1) + generator/correlate (48 per in-band bin);
    pass 2 = N2-point row FFTs (5 N log2 N2) + |z|^2 / peak / threshold (6 N)."""
    return 5.0 * n * lg1 + 48.0 * n_b_mean, 5.0 * n * lg2 + 6.0 * n


def mean_band_bins(wl) -> float:
    """Mean number of in-band bins k_lo..k_hi over the bank (host arithmetic on inputs only)."""
    from testsupport.workloads import T_SUN_S
    mt = wl.bank[:, 0] + wl.bank[:, 1]
    f_isco = 1.0 / (6.0 ** 1.5 * np.pi * mt * T_SUN_S)
    k_lo = math.ceil(wl.f_low * wl.n / wl.fs)
    k_hi = np.minimum(np.floor(f_isco * wl.n / wl.fs), wl.n // 2 - 1)
    return float(np.mean(np.maximum(k_hi - k_lo + 1, 0)))


def cpu_model() -> str:
    """The host CPU as /proc/cpuinfo names it (read at run time)."""
    try:
        with open("/proc/cpuinfo") as fh:
            for ln in fh:
                if ln.lower().startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    import platform
    return platform.processor() or platform.machine()


def oracle_rate(wl, n_sample: int, repeats: int = 1):
    """Time the CPU oracle, as it stands, on the first n_sample templates of the workload."""
    import oracle
    o = oracle.Oracle(wl.n, wl.fs, wl.f_low)
    o.set_psd(wl.psd)
    o.load_segment(wl.samples)
    bank = np.ascontiguousarray(wl.bank[:n_sample])
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        o.filter_bank(bank, wl.threshold)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    o.close()
    return n_sample / best, best, oracle.num_threads()


# --------------------------------------------------------------------------- reference arm
def run_reference(args):
    rank = _env_int("RANK", 0)
    if rank != 0:
        return 0
    import oracle
    wl = make_workload(args.workload, 1, 0)
    cores = oracle.num_threads()
    n_sample = max(1, min(wl.n_templates, 8 * cores))      # eight templates per thread per step (~1 s at N = 2^20)
    o = oracle.Oracle(wl.n, wl.fs, wl.f_low)
    bank = np.ascontiguousarray(wl.bank[:n_sample])
    def step():
        o.set_psd(wl.psd)
        o.load_segment(wl.samples)
        o.filter_bank(bank, wl.threshold)
    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    sample = f"first {n_sample} templates of {wl.name} per step (8 per thread), set_psd + load_segment + filter_bank"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": wl.name, "n": wl.n, "fs_hz": wl.fs, "f_low_hz": wl.f_low,
                   "templates_per_step": n_sample, "threshold": wl.threshold},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "cpu_model": cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------- our arm
def kernel_source_hash() -> str:
    """sha256 over the kernel sources the traffic figure belongs to (csrc/*.cu, *.cuh, include/cbmf.h)."""
    import glob
    import hashlib
    h = hashlib.sha256()
    files = sorted(glob.glob(os.path.join(ROOT, "paper_1006_4644_b200", "csrc", "*.cu*"))) + \
        [os.path.join(ROOT, "include", "cbmf.h")]
    for f in files:
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def load_traffic(n: int):
    """DRAM bytes per template of the two pass kernels from the tracked ncu summary profiles/traffic.json
    (written by `bench.py --traffic-report` from one `ncu --set full` capture).  None unless the capture was taken on
    exactly the kernel sources of this tree (hash) and at this N."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            t = json.load(fh)
    except Exception:
        return None, "profiles/traffic.json missing"
    if t.get("kernel_source_hash") != kernel_source_hash():
        return None, f"profiles/traffic.json was captured on other kernel sources ({t.get('kernel_source_hash')})"
    if int(t.get("n", 0)) != n:
        return None, f"profiles/traffic.json is for n = {t.get('n')}"
    return t, t.get("source", "profiles/traffic.json")


def fp32_probe(device: int):
    """Measured FFMA / FFMA2 TFLOP/s on dependent FMA chains: the library's diagnostic cbmf_debug_fp32_peak."""
    try:
        from paper_1006_4644_b200 import cbmf
        return cbmf.debug_fp32_peak(device)
    except Exception:
        return None, None


def measure(torch, dist, cbmf, wl, dev, local, world, K, Wm, cap, args, with_e2e=True, with_passes=True):
    """All legs of one workload on this rank.  -> dict of raw measurements."""
    B, n = wl.n_templates, wl.n
    stream = torch.cuda.Stream(device=dev)
    out = {}
    with torch.cuda.stream(stream):
        ctx = cbmf.Context(n, wl.fs, wl.f_low, device=local, stream=stream.cuda_stream)
        if args.sub_batch:
            ctx.set_sub_batch(args.sub_batch)
        if args.streams:
            ctx.set_streams(args.streams)
        psd_d = torch.from_numpy(wl.psd).to(dev)
        smp_d = torch.from_numpy(wl.samples).to(dev)
        bank_d = torch.from_numpy(np.ascontiguousarray(wl.bank)).to(dev)
        peaks_d = torch.empty(B * 16, dtype=torch.uint8, device=dev)
        trig_d = torch.empty(cap * 16, dtype=torch.uint8, device=dev)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

        def step_dev():
            ctx.set_psd(psd_d)
            ctx.load_segment(smp_d)
            return ctx.filter_bank_into(bank_d, wl.threshold, peaks_d, trig_d, cap)

        def timed(fn, k):
            """k steps, each bracketed by CUDA events on the context's stream; L2 flushed
            (untimed) before every step.  -> (sum of step times in ms, last result)"""
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(k)]
            res = None
            for i in range(k):
                flush.fill_(i & 0xFF)
                evs[i][0].record(stream)
                res = fn()
                evs[i][1].record(stream)
            stream.synchronize()
            return sum(a.elapsed_time(b) for a, b in evs), res

        def barrier():
            if world > 1:
                dist.barrier()
            torch.cuda.synchronize()

        def max_over_ranks(x):
            t = torch.tensor([x], dtype=torch.float64, device=dev)
            if world > 1:
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())

        # ---- device-resident leg: `value`
        for _ in range(Wm):
            flush.fill_(1)
            step_dev()
        barrier()
        l0 = ctx.launch_count()
        with ClockSampler(local) as clk:
            ms_total, (nf, rc) = timed(step_dev, K)
        barrier()
        out["launches"] = ctx.launch_count() - l0
        out["ms_max"] = max_over_ranks(ms_total)
        out["clocks"] = clk.summary()
        out["nf"] = int(nf)
        out["split"] = ctx.get_split()
        out["sub_batch"], out["streams"] = ctx.get_sub_batch(), ctx.get_streams()
        out["peaks"] = peaks_d.cpu().numpy().view(cbmf.PEAK_DTYPE).copy()

        # ---- roofline legs: per-launch events inside K more steps, every launch alone (mode 1) and in the
        # real overlapped schedule (mode 2)
        if with_passes:
            for mode, key in ((1, "alone"), (2, "overlapped")):
                ctx.set_profiling(mode)
                p_ms, p_n = [0.0, 0.0], [0, 0]
                for i in range(K):
                    flush.fill_(i & 0xFF)
                    step_dev()
                    for w in (0, 1):
                        ms, nl = ctx.last_pass_time(w)
                        p_ms[w] += ms
                        p_n[w] += nl
                ctx.set_profiling(0)
                out["pass_" + key] = (p_ms, p_n)

        # ---- e2e leg: host-pointer entry points, pinned host buffers
        if with_e2e:
            psd_h = torch.from_numpy(wl.psd).pin_memory()
            smp_h = torch.from_numpy(wl.samples).pin_memory()
            bank_h = torch.from_numpy(np.ascontiguousarray(wl.bank)).pin_memory()
            peaks_h = torch.empty(B * 16, dtype=torch.uint8).pin_memory()
            trig_h = torch.empty(cap * 16, dtype=torch.uint8).pin_memory()

            def step_host():
                ctx.set_psd(psd_h)
                ctx.load_segment(smp_h)
                return ctx.filter_bank_into(bank_h, wl.threshold, peaks_h, trig_h, cap)

            for _ in range(Wm):
                step_host()
            barrier()
            e_ms, (nf_h, rc_h) = timed(step_host, K)
            barrier()
            out["e_ms_max"] = max_over_ranks(e_ms)
            # the same step with the host-side reduction of PAPER.md:103 behind it, clustered while the GPU filters
            # the following sub-batches: must not cost anything
            ev_h = torch.empty(cap * 16, dtype=torch.uint8).pin_memory()

            def step_host_clustered():
                ctx.set_psd(psd_h)
                ctx.load_segment(smp_h)
                return ctx.filter_bank_clustered_into(bank_h, wl.threshold, args.cluster_window, peaks_h, ev_h, cap)

            for _ in range(Wm):
                step_host_clustered()
            barrier()
            c_ms, (n_ev, nf_c, rc_c) = timed(step_host_clustered, K)
            barrier()
            out["c_ms_max"] = max_over_ranks(c_ms)
            out["n_events"] = int(n_ev)
            # the paper's own template path (NEXT-3: time-domain generation, forward FFT, normalisation by a
            # reduction, product, inverse FFT -- every intermediate in device memory) on a bounded sample
            if args.workload == "cfg1" and world == 1:
                n_td = min(B, 128)
                bank_td = np.ascontiguousarray(wl.bank[:n_td])
                ctx.load_segment(smp_h)
                ctx.filter_bank_td(bank_td, wl.threshold)                      # warm-up (allocations)
                a_ev, b_ev = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a_ev.record(stream)
                for _ in range(3):
                    ctx.filter_bank_td(bank_td, wl.threshold)
                b_ev.record(stream)
                stream.synchronize()
                out["td_us_per_template"] = 1e3 * a_ev.elapsed_time(b_ev) / (3 * n_td)
                out["td_templates"] = n_td
            out["h2d"] = psd_h.numel() * 8 + smp_h.numel() * 4 + bank_h.numel() * 8
            # what the three host-pointer calls copy back (csrc/cbmf.cu): the 8-byte input-check word of set_psd and of
            # load_segment; filter_bank's 32-byte status block, the peaks and its trigger staging block, which is
            # min(capacity, 4096) records whatever the count; a bank with more triggers than that block holds goes
            # through the general collection: the kept triggers and the peaks once more
            n_fast = min(cap, 4096)
            out["d2h"] = 8 + 8 + 32 + B * 16 + n_fast * 16
            if nf_h > n_fast:
                out["d2h"] += min(nf_h, cap) * 16 + B * 16
        ctx.close()
    return out


# PAPER.md:249-254, table 4.1: vector size, low-frequency cut, max templates processed in real time (GTX 275)
PAPER_ONLINE = ((18, 30.0, 3435), (19, 23.0, 4095), (20, 15.0, 4478), (21, 14.0, 4279))


def online_capacity(torch, cbmf, local, n_templates=2048, n_segments=4):
    """NEXT-2: the paper's online figure through cbmf_filter_stream: [1.4, 1.4] Msun templates,
    fs = 4096 Hz, the paper's vector sizes and cut-offs, segments overlapping by half (what its table implies:
    4478 = 128 s / 28.6 ms at 2^20); capacity = templates that fit into the hop time of one segment."""
    from testsupport import workloads as W
    fs, rows = 4096.0, []
    for log2n, f_low, paper in PAPER_ONLINE:
        n = 1 << log2n
        hop = n // 2
        n_total = n + (n_segments - 1) * hop
        big = 1 << int(math.ceil(math.log2(n_total)))
        psd_big = W.onesided_psd("A", big, fs, f_low)
        stream = W.to_time_domain(W.noise_spectrum(big, fs, f_low, psd_big, 900 + log2n), big, fs)[:n_total]
        stream_h = torch.from_numpy(np.ascontiguousarray(stream)).pin_memory()
        bank = W.draw_bank(910 + log2n, n_templates, 1.35, 1.45)
        st = torch.cuda.Stream(device=torch.device("cuda", local))
        with torch.cuda.stream(st):
            ctx = cbmf.Context(n, fs, f_low, device=local, stream=st.cuda_stream)
            ctx.set_psd(W.onesided_psd("A", n, fs, f_low))
            ctx.filter_stream(stream_h, bank, 6.0, hop)                       # warm-up
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(st)
            pk, tr, offs, nf, rc = ctx.filter_stream(stream_h, bank, 6.0, hop)
            b.record(st)
            st.synchronize()
            ms_seg = a.elapsed_time(b) / n_segments
            ctx.close()
        rows.append({"n_log2": log2n, "f_low_hz": f_low, "hop_s": hop / fs, "templates": n_templates, "segments": n_segments,
                     "ms_per_segment": ms_seg, "us_per_template": 1e3 * ms_seg / n_templates,
                     "max_templates_in_real_time": int(n_templates * (hop / fs) / (ms_seg * 1e-3)),
                     "paper_gtx275": paper, "triggers": int(nf)})
    return rows


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start the N ranks ourselves
    (one process per GPU, rendezvous on 127.0.0.1) and pass rank 0's line through."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1006_4644_b200 import cbmf

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)
    rank, world, local = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1), _env_int("LOCAL_RANK", 0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    wl = make_workload(args.workload, world, rank)
    B, n = wl.n_templates, wl.n
    cap = args.trig_capacity
    K, Wm = args.steps, args.warmup
    m = measure(torch, dist, cbmf, wl, dev, local, world, K, Wm, cap, args)
    ms_max = m["ms_max"]
    value = B * world * K / (ms_max * 1e-3)
    e_value = B * world * K / (m["e_ms_max"] * 1e-3)
    fp32_meas = fp32_probe(local) if rank == 0 else (None, None)

    # ---- sustained record: a few steps of configs[2] (65 536 templates, ~0.2 s per step): the state a
    # 1-2 million-template bank runs in, with its own clocks
    sustained = None
    if args.workload == "cfg1" and not args.no_sustained:
        wl2 = make_workload("cfg2", world, rank)
        Ks = max(2, min(K, args.sustained_steps))
        m2 = measure(torch, dist, cbmf, wl2, dev, local, world, Ks, 3, 1 << 20, args, with_e2e=False, with_passes=False)
        lg1s, lg2s = m2["split"]
        f1s, f2s = pass_flops(wl2.n, lg1s, lg2s, mean_band_bins(wl2))
        v2 = wl2.n_templates * world * Ks / (m2["ms_max"] * 1e-3)
        sustained = {
            "workload": "cfg2", "templates_per_step_per_gpu": wl2.n_templates, "steps": Ks, "warmup": 3,
            "value": v2, "unit": UNIT, "ms_per_step": m2["ms_max"] / Ks, "clocks": m2["clocks"],
            "gpu_launches": int(m2["launches"]), "triggers_found": m2["nf"],
            "whole_path": {"flops_per_template": f1s + f2s, "us_per_template": 1e3 * m2["ms_max"] / (wl2.n_templates * Ks),
                           "frac_of_fp32_peak": (f1s + f2s) * v2 / world / 1e12 / FP32_PEAK_TFLOPS,
                           "dense_equivalent_frac": (5.0 * wl2.n * (lg1s + lg2s) + 6.0 * wl2.n + 48.0 * (wl2.n / 2)) * v2 / world / 1e12 / FP32_PEAK_TFLOPS,
                           "note": "frac_of_fp32_peak counts the generator on the in-band bins only (mean n_b/N = 0.10 in cfg2); "
                                   "dense_equivalent_frac counts it on all N/2 bins (SURVEY.md §8(d))"},
        }

    online = online_capacity(torch, cbmf, local) if (world == 1 and args.workload == "cfg1" and not args.no_online) else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline numbers for the dominant pass (FFT split as the library chose it)
    lg1, lg2 = m["split"]
    n_b = mean_band_bins(wl)
    f1, f2 = pass_flops(n, lg1, lg2, n_b)
    p_ms, p_n = m["pass_alone"]
    o_ms, o_n = m["pass_overlapped"]
    which = 0 if p_ms[0] >= p_ms[1] else 1
    avg_launch_ms = p_ms[which] / max(p_n[which], 1)
    tmpl_per_launch = B * K / max(p_n[which], 1)
    flops_launch = (f1, f2)[which] * tmpl_per_launch
    achieved = flops_launch / (avg_launch_ms * 1e-3) / 1e12
    peaks_file = {}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            peaks_file = json.load(fh)
    except Exception:
        pass
    traffic, traffic_src = load_traffic(n)
    tr_per_tmpl = None if traffic is None else traffic["dram_bytes_per_template"][which]
    roofline = {
        "bound": "alu", "kernel": ("p1_kernel (SPA generate + correlate + column FFT)",
                                   "p2_kernel (twiddle + row FFT + |z|^2 + arg-max/threshold)")[which],
        "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP32_PEAK_TFLOPS,
        "peak_source": "148 SM x 128 FP32 lanes x 2 x 1.965 GHz (B200_PROFILING.md unit counts and clocks; DESIGN.md §6)",
        "peak_measured_tflops": fp32_meas[1],          # packed-FFMA2 chains on every SM (the cross-check)
        "peak_measured_ffma_tflops": fp32_meas[0],
        "frac_of_measured_peak": (achieved / fp32_meas[1]) if fp32_meas[1] else None,
        "traffic": None if tr_per_tmpl is None else tr_per_tmpl * tmpl_per_launch,
        "traffic_source": traffic_src,
        "algorithmic_bytes_per_launch": 8.0 * n * tmpl_per_launch,
        "flops_per_launch": flops_launch, "avg_launch_ms": avg_launch_ms, "templates_per_launch": tmpl_per_launch,
        "pass_ms_per_step": [p_ms[0] / K, p_ms[1] / K],
        "pass_launch_ms_overlapped": [o_ms[0] / max(o_n[0], 1), o_ms[1] / max(o_n[1], 1)],
        "note": ("`achieved` and pass_ms_per_step are taken with every launch ALONE on the GPU (one stream); in the timed "
                 "schedule four launch pairs are in flight and the long-lived pass-1 blocks share the SMs with pass-2 blocks "
                 "of the other pairs, so the passes overlap (pass_launch_ms_overlapped: mean duration of a launch in that "
                 "schedule, events on its own stream); whole_path gives the fraction of the FP32 peak reached by the whole step"),
        "whole_path": {
            "flops_per_template": f1 + f2, "us_per_template": 1e3 * ms_max / (B * K),
            "achieved_tflops": (f1 + f2) * B * K / (ms_max * 1e-3) / 1e12,
            "frac_of_fp32_peak": (f1 + f2) * B * K / (ms_max * 1e-3) / 1e12 / FP32_PEAK_TFLOPS,
            "inter_pass_bytes_per_template": 16 * n,
            "hbm_gbs_measured_peak": peaks_file.get("hbm_gbs"),
            "hbm_frac_if_y_spills": (16.0 * n * value / world / 1e9 / peaks_file["hbm_gbs"]) if peaks_file.get("hbm_gbs") else None,
        },
    }

    # ---- CPU oracle on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu:
        import oracle
        cores = oracle.num_threads()
        n_sample = min(B, max(64, 16 * cores))         # ~0.1 core-second per template at N = 2^20
        v, secs, cores = oracle_rate(wl, n_sample)
        # one thread, mean over >= 8 templates (the paper compares with ONE core)
        n_one = min(B, 8)
        oracle.set_num_threads(1)
        try:
            v1, secs1, _ = oracle_rate(wl, n_one)
        finally:
            oracle.set_num_threads(cores)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {n_sample} templates of {wl.name}, filter_bank only, {secs:.2f} s wall",
               "single_thread": {"value": v1, "unit": UNIT, "cores": 1, "ms_per_template": 1e3 * secs1 / n_one,
                                 "sample": f"first {n_one} templates of {wl.name}, filter_bank only, {secs1:.2f} s wall"},
               "cpu_model": cpu_model()}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": wl.name, "n": n, "fs_hz": wl.fs, "f_low_hz": wl.f_low,
                   "templates_per_step_per_gpu": B, "threshold": wl.threshold, "sub_batch": m["sub_batch"],
                   "streams": m["streams"], "fft_split_log2": [lg1, lg2],
                   "l2": "flushed (256 MiB fill) before every timed step",
                   "step": "set_psd + load_segment + filter_bank (S0-S8)",
                   "parallelism": f"bank sharded over {world} GPU(s), segment replicated"},
        "segment_seconds_per_wall_second": (n / wl.fs) / (ms_max / K * 1e-3),
        "triggers_found": m["nf"], "peak_snr_max": float(m["peaks"]["snr_max"].max()),
        "e2e": {"value": e_value, "unit": UNIT, "h2d_bytes_per_step": int(m["h2d"]), "d2h_bytes_per_step": int(m["d2h"])},
        "e2e_clustered": {"value": B * world * K / (m["c_ms_max"] * 1e-3), "unit": UNIT, "events": m["n_events"],
                          "window_samples": args.cluster_window,
                          "what": "cbmf_filter_bank_clustered: raw triggers reduced to events on the host while the GPU "
                                  "filters the next sub-batches (NEXT-1, PAPER.md:103, :131)"},
        "paper_path": None if "td_us_per_template" not in m else {
            "us_per_template": m["td_us_per_template"], "value": 1e6 / m["td_us_per_template"], "unit": UNIT,
            "templates": m["td_templates"],
            "what": "cbmf_filter_bank_td: the paper's own per-template pipeline on the same GPU (time-domain generation of two "
                    "polarisations, forward FFT, normalisation by a reduction, product, inverse FFT, every intermediate in "
                    "device memory: PAPER.md:127-131, :177-179; 28 ms per template on the paper's GTX 275, PAPER.md:231) -- "
                    "the comparison path, not the product's"},
        "gpu_launches": int(m["launches"]),
        "clocks": m["clocks"],
        "roofline": roofline,
        "sustained": sustained,
        "online_capacity": online,
        "cpu_baseline": cpu,
    }
    # the second bound of the whole step: the inter-pass buffer Y goes through HBM once each way (16 N bytes per
    # template: ncu reads 16.6 MB at N = 2^20, profiles/); the regime is the bound the step sits closer to
    hbm_peak = peaks_file.get("hbm_gbs")
    hbm_gbs = 16.0 * n * value / world / 1e9
    alu_frac = roofline["whole_path"]["frac_of_fp32_peak"]
    roofline["hbm"] = {"bytes_per_template": 16 * n, "achieved_gbs": hbm_gbs, "peak": hbm_peak, "unit": "GB/s",
                       "frac": (hbm_gbs / hbm_peak) if hbm_peak else None,
                       "peak_source": "MEASURED_PEAKS.json hbm_gbs" if hbm_peak else "MEASURED_PEAKS.json missing"}
    roofline["regime"] = ("hbm" if (hbm_peak and hbm_gbs / hbm_peak > alu_frac) else "alu")
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


# --------------------------------------------------------------------------- configs[4]: the kernel sweep
# Segment lengths N = 2^16 .. 2^24 x template batch sizes 1 / 8 / 64 / 512, fs = 4096 Hz, f_low = 40 Hz, PSD of
# config 0, m1, m2 uniform in [1, 3] Msun (BASELINE.json configs[4]).  For every point, on one GPU,
# device-resident data:
#   ifft      the hand-written batched inverse FFT alone (cbmf_debug_ifft_dev: pass 1 + pass 2 with plain load /
#             store epilogues) on random complex input, out of place
#   cufft     the same transform by cuFFT (torch.fft.ifft, norm="forward" = unnormalised) -- the comparison
#             baseline only; cuFFT is never on the product path
#   generate  the SPA generator alone writing q~ = w e^{i Psi} to HBM (cbmf_debug_generate_dev)
#   filter    the whole hot path (cbmf_filter_bank_dev: S2-S8) in templates/s
#     python bench.py --workload cfg4 [--log2n 16 ... 24] [--batches 1 8 64 512] [--repeats 5] [--markdown]
# One JSON line per point on stdout (not the driver's bench line: that is cfg1); --markdown prints a table instead.
# Points whose buffers would exceed --max-gib (input + output of the FFT comparison) run with the largest batch
# that fits and say so in "batch_run".
def _sweep_time(fn, stream, repeats):
    import torch
    fn()
    stream.synchronize()
    best = None
    for _ in range(repeats):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        fn()
        b.record(stream)
        stream.synchronize()
        ms = a.elapsed_time(b)
        best = ms if best is None else min(best, ms)
    return best


def sweep_point(log2n: int, batch: int, repeats: int, max_gib: float):
    import torch
    from paper_1006_4644_b200 import cbmf
    from testsupport import workloads as W
    n = 1 << log2n
    dev = torch.device("cuda", 0)
    stream = torch.cuda.Stream(device=dev)
    b_run = batch
    while b_run > 1 and 2 * 8 * n * b_run > max_gib * (1 << 30):
        b_run //= 2
    wl = W.sweep_point(log2n, batch)
    out = {"log2n": log2n, "batch": batch, "batch_run": b_run}
    with torch.cuda.stream(stream):
        ctx = cbmf.Context(n, wl.fs, wl.f_low, device=0, stream=stream.cuda_stream)
        ctx.set_psd(wl.psd)
        ctx.load_segment(wl.samples)
        g = torch.Generator(device=dev).manual_seed(1000 + log2n)
        x = torch.view_as_complex(torch.randn(b_run, n, 2, generator=g, device=dev, dtype=torch.float32))
        y = torch.empty_like(x)
        ms_h = _sweep_time(lambda: ctx.debug_ifft(x, y), stream, repeats)
        # torch adds an element-wise pass of its own behind the library transform when it is given `out=` (ncu shows
        # it); the comparison figure is the faster of the two ways of calling it
        ms_c = min(_sweep_time(lambda: torch.fft.ifft(x, dim=1, norm="forward", out=y), stream, repeats),
                   _sweep_time(lambda: torch.fft.ifft(x, dim=1, norm="forward"), stream, repeats))
        ref = torch.fft.ifft(x[:1], dim=1, norm="forward")
        got = ctx.debug_ifft(x[:1].contiguous())
        err = float((got - ref).abs().max() / ref.abs().max())
        flops = 5.0 * n * log2n * b_run
        out.update(ifft_ms=ms_h, cufft_ms=ms_c, ifft_vs_cufft=ms_c / ms_h, ifft_gflops=flops / ms_h / 1e6,
                   cufft_gflops=flops / ms_c / 1e6, ifft_max_rel_diff_vs_cufft=err)
        del x, y
        bank = torch.from_numpy(np.ascontiguousarray(wl.bank[:b_run])).to(dev)
        q = torch.empty(b_run * (n // 2), dtype=torch.complex64, device=dev)
        ms_g = _sweep_time(lambda: ctx.debug_generate_dev(bank, q), stream, repeats)
        out.update(generate_ms=ms_g, generate_gbins_per_s=b_run * (n // 2) / ms_g / 1e6)
        del q
        bank_full = torch.from_numpy(np.ascontiguousarray(wl.bank)).to(dev)
        peaks = torch.empty(batch * 16, dtype=torch.uint8, device=dev)
        trig = torch.empty((1 << 16) * 16, dtype=torch.uint8, device=dev)
        ms_f = _sweep_time(lambda: ctx.filter_bank_into(bank_full, wl.threshold, peaks, trig, 1 << 16), stream, repeats)
        out.update(filter_ms=ms_f, filter_templates_per_s=batch / ms_f * 1e3,
                   filter_us_per_template=ms_f * 1e3 / batch)
        ctx.close()
    return out


def run_cfg4(a):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --workload cfg4: no CUDA device -- the product path has no CPU fallback")
    rows = []
    for l in a.log2n:
        for b in a.batches:
            r = sweep_point(l, b, a.repeats, a.max_gib)
            rows.append(r)
            if not a.markdown:
                print(json.dumps(r), flush=True)
    if a.markdown:
        print("| log2 N | batch (run) | hand IFFT ms | cuFFT ms | cuFFT / hand | hand GFLOP/s | generator Gbin/s | "
              "filter templates/s | filter us/template |")
        print("|---:|---:|---:|---:|---:|---:|---:|---:|---:|")
        for r in rows:
            print(f"| {r['log2n']} | {r['batch']} ({r['batch_run']}) | {r['ifft_ms']:.4f} | {r['cufft_ms']:.4f} | "
                  f"{r['ifft_vs_cufft']:.2f} | {r['ifft_gflops']:.0f} | {r['generate_gbins_per_s']:.1f} | "
                  f"{r['filter_templates_per_s']:.0f} | {r['filter_us_per_template']:.2f} |")
    return 0


# --------------------------------------------------------------------------- profiles/traffic.json
# One `ncu --set full` capture of the two FFT-pass kernels -> the tracked summary profiles/traffic.json that
# `roofline.traffic` is read from.  On the GPU box, in the same gpurun command as the capture (stamps the kernel
# sources the capture ran on):      python bench.py --traffic-stamp > gpurun_out/src_hash.txt
# Here (ncu reads reports without a GPU):
#     python bench.py --traffic-report gpurun_out/prof.ncu-rep --traffic-stamp-file gpurun_out/src_hash.txt \
#         --traffic-templates-per-launch 256 --traffic-command "<the ncu command line>"
# dram bytes per template = (dram__bytes_read.sum + dram__bytes_write.sum) of a launch / templates per launch,
# averaged over the captured launches of each kernel.
def write_traffic(a):
    import csv
    import io
    import subprocess
    stamp = open(a.stamp_file).read().strip() if a.stamp_file else kernel_source_hash()
    raw = subprocess.run(["ncu", "-i", a.report, "--page", "raw", "--csv"], check=True, capture_output=True, text=True).stdout
    rows = list(csv.reader(io.StringIO(raw)))
    hdr = rows[0]
    col = {name: i for i, name in enumerate(hdr)}
    per = {"p1_kernel": [], "p2_kernel": []}
    dur = {"p1_kernel": [], "p2_kernel": []}
    for r in rows[2:]:                       # row 1 holds the units
        name = r[col["Kernel Name"]]
        for k in per:
            if k in name:
                rd = float(r[col["dram__bytes_read.sum"]].replace(",", ""))
                wr = float(r[col["dram__bytes_write.sum"]].replace(",", ""))
                unit_r = rows[1][col["dram__bytes_read.sum"]]
                unit_w = rows[1][col["dram__bytes_write.sum"]]
                scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
                per[k].append(rd * scale.get(unit_r, 1.0) + wr * scale.get(unit_w, 1.0))
                d = float(r[col["gpu__time_duration.sum"]].replace(",", ""))
                dur[k].append(d * {"ns": 1e-3, "us": 1.0, "ms": 1e3}.get(rows[1][col["gpu__time_duration.sum"]], 1.0))
    out = {
        "kernel_source_hash": stamp, "n": a.n, "templates_per_launch": a.templates_per_launch,
        "launches_captured": [len(per["p1_kernel"]), len(per["p2_kernel"])],
        "dram_bytes_per_template": [sum(v) / len(v) / a.templates_per_launch if v else None for v in (per["p1_kernel"], per["p2_kernel"])],
        "gpu_time_us_per_launch_under_ncu": [sum(v) / len(v) if v else None for v in (dur["p1_kernel"], dur["p2_kernel"])],
        "source": f"ncu --set full, {os.path.basename(a.report)} (profiles/traffic.json)", "command": a.command,
    }
    with open(a.out, "w") as fh:
        json.dump(out, fh, indent=1)
        fh.write("\n")
    print(json.dumps(out))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=["cfg1", "cfg2", "cfg3", "cfg4"], default="cfg1",
                    help="cfg4 = the configs[4] kernel sweep (one JSON line per point; not the driver's bench line)")
    ap.add_argument("--log2n", type=int, nargs="*", default=list(range(16, 25)), help="cfg4: segment lengths")
    ap.add_argument("--batches", type=int, nargs="*", default=[1, 8, 64, 512], help="cfg4: templates per point")
    ap.add_argument("--repeats", type=int, default=5, help="cfg4: timed repeats per measurement (best of)")
    ap.add_argument("--max-gib", type=float, default=16.0, help="cfg4: cap on the FFT comparison buffers")
    ap.add_argument("--markdown", action="store_true", help="cfg4: print a table instead of JSON lines")
    ap.add_argument("--traffic-stamp", action="store_true", help="print the hash of the kernel sources and exit")
    ap.add_argument("--traffic-report", dest="report", help="ncu report to turn into profiles/traffic.json")
    ap.add_argument("--traffic-stamp-file", dest="stamp_file")
    ap.add_argument("--traffic-n", dest="n", type=int, default=1 << 20)
    ap.add_argument("--traffic-templates-per-launch", dest="templates_per_launch", type=int, default=256)
    ap.add_argument("--traffic-command", dest="command", default="")
    ap.add_argument("--traffic-out", dest="out", default=os.path.join(ROOT, "profiles", "traffic.json"))
    ap.add_argument("--sub-batch", type=int, default=0, help="templates per launch pair (0 = library default)")
    ap.add_argument("--streams", type=int, default=0, help="launch pairs in flight (0 = library default)")
    ap.add_argument("--trig-capacity", type=int, default=1 << 16)
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--cluster-window", type=int, default=64, help="event window in samples for the e2e_clustered leg")
    ap.add_argument("--no-online", action="store_true", help="skip the online_capacity record (cbmf_filter_stream, PAPER.md table 4.1)")
    ap.add_argument("--no-sustained", action="store_true", help="skip the cfg2 `sustained` record of the default run")
    ap.add_argument("--sustained-steps", type=int, default=3)
    args = ap.parse_args()
    if args.traffic_stamp:
        print(kernel_source_hash())
        return 0
    if args.report:
        return write_traffic(args)
    if args.workload == "cfg4":
        return run_cfg4(args)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
