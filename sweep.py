"""Kernel sweep of BASELINE.json configs[4]: segment lengths N = 2^16 .. 2^24
x template batch sizes 1 / 8 / 64 / 512, fs = 4096 Hz, f_low = 40 Hz, PSD of config 0,
m1, m2 uniform in [1, 3] Msun.  For every point, on one GPU, device-resident data:

  ifft      the hand-written batched inverse FFT alone (cbmf_debug_ifft_dev: pass 1 + pass 2 with
            plain load / store epilogues) on random complex input, out of place
  cufft     the same transform by cuFFT (torch.fft.ifft, norm="forward" = unnormalised) -- the
            comparison baseline only; cuFFT is never on the product path
  generate  the SPA generator alone writing q~ = w e^{i Psi} to HBM (cbmf_debug_generate_dev)
  filter    the whole hot path (cbmf_filter_bank_dev: S2-S8) in templates/s

    python sweep.py [--log2n 16 ... 24] [--batches 1 8 64 512] [--repeats 5]

One JSON line per point on stdout; `--markdown` prints a table instead.  Points whose buffers
would exceed --max-gib (input + output of the FFT comparison) run with the largest batch that fits
and say so in "batch_run".
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _time(fn, stream, repeats):
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


def run_point(log2n: int, batch: int, repeats: int, max_gib: float):
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
        ms_h = _time(lambda: ctx.debug_ifft(x, y), stream, repeats)
        # torch adds an element-wise pass of its own behind the library transform when it is given `out=` (ncu shows
        # it); the comparison figure is the faster of the two ways of calling it
        ms_c = min(_time(lambda: torch.fft.ifft(x, dim=1, norm="forward", out=y), stream, repeats),
                   _time(lambda: torch.fft.ifft(x, dim=1, norm="forward"), stream, repeats))
        ref = torch.fft.ifft(x[:1], dim=1, norm="forward")
        got = ctx.debug_ifft(x[:1].contiguous())
        err = float((got - ref).abs().max() / ref.abs().max())
        flops = 5.0 * n * log2n * b_run
        out.update(ifft_ms=ms_h, cufft_ms=ms_c, ifft_vs_cufft=ms_c / ms_h, ifft_gflops=flops / ms_h / 1e6,
                   cufft_gflops=flops / ms_c / 1e6, ifft_max_rel_diff_vs_cufft=err)
        del x, y
        bank = torch.from_numpy(np.ascontiguousarray(wl.bank[:b_run])).to(dev)
        q = torch.empty(b_run * (n // 2), dtype=torch.complex64, device=dev)
        ms_g = _time(lambda: ctx.debug_generate_dev(bank, q), stream, repeats)
        out.update(generate_ms=ms_g, generate_gbins_per_s=b_run * (n // 2) / ms_g / 1e6)
        del q
        bank_full = torch.from_numpy(np.ascontiguousarray(wl.bank)).to(dev)
        peaks = torch.empty(batch * 16, dtype=torch.uint8, device=dev)
        trig = torch.empty((1 << 16) * 16, dtype=torch.uint8, device=dev)
        ms_f = _time(lambda: ctx.filter_bank_into(bank_full, wl.threshold, peaks, trig, 1 << 16), stream, repeats)
        out.update(filter_ms=ms_f, filter_templates_per_s=batch / ms_f * 1e3,
                   filter_us_per_template=ms_f * 1e3 / batch)
        ctx.close()
    return out


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--log2n", type=int, nargs="*", default=list(range(16, 25)))
    ap.add_argument("--batches", type=int, nargs="*", default=[1, 8, 64, 512])
    ap.add_argument("--repeats", type=int, default=5)
    ap.add_argument("--max-gib", type=float, default=16.0)
    ap.add_argument("--markdown", action="store_true")
    a = ap.parse_args(argv)
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("sweep: no CUDA device -- the product path has no CPU fallback")
    rows = []
    for l in a.log2n:
        for b in a.batches:
            r = run_point(l, b, a.repeats, a.max_gib)
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


if __name__ == "__main__":
    sys.exit(main())
