"""Per-config timings for the five BASELINE.json workloads (bench.py times only the headline one).

  python -m paper_2606_23698_b200.bench_configs [--reps 5]

For each config: ms per transform (CUDA events on the current stream, median of reps after 3 warm-ups),
5 N log2 N GFLOP/s, fraction of the HBM roof (algorithmic bytes = 32 B per element per axis pass over the
measured copy bandwidth), cuFFT Z2Z fp64 on the same tensor for context.  Inputs are the seeded recipes of
inputs.CONFIGS, generated on the host.  One JSON line per config.
"""
import argparse
import json
import math
import os

import torch

from . import inputs, ozfft

_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _time(fn, reps):
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    ts.sort()
    return ts[len(ts) // 2], ts[0]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--reps", type=int, default=5)
    args = ap.parse_args()
    try:
        hbm = float(json.load(open(os.path.join(_ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        hbm = 6650.0
    for name, (kind, shape, dist, seed) in inputs.CONFIGS.items():
        h = torch.empty(shape, dtype=torch.complex128)
        if dist == "uniform":
            inputs.uniform_pm1(shape, seed, out=h.numpy())
        else:
            h.copy_(torch.from_numpy(inputs.make(dist, shape, seed)))
        x = h.cuda()
        y = torch.empty_like(x)
        if kind == "3d":
            plan = ozfft.Plan(*shape)
            flop = 5.0 * x.numel() * math.log2(x.numel())
            passes = 3
            cufft = lambda: torch.fft.fftn(x)
        else:
            plan = ozfft.Plan.batched_1d(shape[1], shape[0])
            flop = 5.0 * x.numel() * math.log2(shape[1])
            passes = 1
            cufft = lambda: torch.fft.fft(x, dim=1)
        med, best = _time(lambda: plan.exec(x, y), args.reps)
        try:
            cmed, _ = _time(cufft, args.reps)
        except Exception:
            cmed = None
        roof_ms = 32.0 * x.numel() * passes / (hbm * 1e9) * 1e3
        print(json.dumps({"config": name, "shape": list(shape), "input": dist, "seed": seed, "launches": plan.num_launches,
                          "ms_median": med, "ms_best": best, "gflops_5NlogN": flop / (med * 1e-3) / 1e9,
                          "hbm_roof_ms": roof_ms, "frac_of_hbm_roof": roof_ms / med, "cufft_z2z_ms": cmed}), flush=True)
        plan.destroy()
        del x, y, h
        torch.cuda.empty_cache()


if __name__ == "__main__":
    main()
